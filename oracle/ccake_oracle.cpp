/*
 * oracle/ccake_oracle.cpp — CPU ORACLE.  TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * A plain, slow, fp64 restatement of one Runge-Kutta (sub)step of the CCAKE 2.0 SPH fluid solver, written from
 * PAPER.md (arxiv 2511.22852) and the readings of DESIGN.md §"Readings".  It follows the paper's order and
 * notation:
 *   Step 0  state and geometry            PAPER.md:164-169 (notation), :482-488 (§4.2), Eq. 85 :954
 *   Step 1  neighbours                    :1434 (§5.9.1), Eq. 78 :915, Eq. 134 :1224
 *   Step 2  smoothing sums                Eq. 68 :864, Eq. 71-72 :877-882, Eq. 77 :910
 *   Step 3  equation of state             Eq. A.5-A.7 :2115-2122, Eq. A.11-A.15 :2136-2156; table :583-593
 *   Step 4  gradient sums                 Eq. 79 :920, Eq. 81-82 :934-938 (Eq. 83 is garbled, DESIGN reading 3)
 *   Step 5  equations of motion           Eq. 38-44 :623-649, Eq. 49-51 :676-680, Eq. 52 :689-693,
 *                                         Eq. 87-104 :964-1041
 *   Step 6  integrator                    not in the paper (DESIGN reading 7): RK2 midpoint / classical RK4
 *   Step 7  conserved totals              §5.6.5 :1049-1063
 *   extra   applicability diagnostics     Eq. 58-61 :797-805 (Kn_pi, Re_pi^-1, Kn_Pi, Re_Pi^-1; pinned on Bjorken)
 *   extra   source smearing               Eq. 35 :521 (pinned: single parton, partition of unity, window, linearity)
 *   extra   source terms I^nu, I_q        Eq. 38 :623, Eq. 42-44 :645-649, Eq. 96 :1003 (pinned: heating and push of a
 *                                         uniform fluid, Bjorken ODE with a source, energy balance of a moving fluid,
 *                                         exact momentum / charge balance)
 *   extra   freeze-out surface element    Eq. 145-148 :1466-1482 (d_mu eps, n_mu, |d sigma|; pinned on Bjorken, Gubser)
 *   extra   offline inverter, forward table :576-593, DESIGN reading 21 (pinned: affine map vs a linear solve, an independent
 *                                         multilinear interpolator, second-order convergence to the exact inversion, backup EoS)
 *
 * There is no blocking, fusion or reordering: loops are gather form (for a { for b }), the per-particle linear
 * system in the unknown time derivatives is written LITERALLY in covariant form with generic 4x4 metric and
 * Christoffel arrays on affine numbers (constant + coefficient per unknown) and solved by dense Gaussian
 * elimination with partial pivoting (Eq. 92-95 :978-988 state that the system is linear; the hand reduction of
 * Eq. 95 is what the CUDA library does, not this file).
 *
 * Parity pins (tests/test_oracle_*.py): kernel normalisation and gradient (Eq. 63, 77, 79), brute-force
 * neighbour lists, partition of unity, conformal EoS identities and round trip (App. A), table exactness for
 * multilinear functions, pairwise momentum/charge conservation, dS/dx0 = dN_q/dx0 = 0 for ideal flow (Eq. 105-106),
 * ideal Gubser flow (Eq. 116-120), Bjorken ideal/shear/bulk ODEs, viscous Gubser ODE (Eq. 112), RK order;
 * tests/test_oracle_pins_dissipative.py: every DNMR second-order term (boost-invariant DNMR ODEs in 2+1D and 3+1D,
 * hand-evaluated tensors on a linear flow and on a rotating disc), the moving-frame part of diffusion (Lorentz
 * covariance of a fluid with a transverse gradient, Christoffel term on the Bjorken slab, normal modes of a boosted
 * fluid), the hyperbolic energy and work totals (energy-momentum conservation, static fluid in hyperbolic
 * coordinates) and the (div v) accumulator (finite difference of sigma*).  A mutation run (19 single-line changes of
 * those terms) is caught by these tests.
 * PARITY UNPINNED: none of the terms on the path; the bulk sector has only the boost-invariant ODEs (the
 * paper itself has no other analytic check for bulk, :1051).
 *
 * Build: g++ -O2 -ffp-contract=off -fopenmp -shared -fPIC (oracle/build.py).  OpenMP is used only as
 * "parallel for" over the particle index a of gather loops, so results do not depend on the thread count.
 */
#include "oracle.h"

#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

namespace {

constexpr int NQ = 3;
constexpr int NUMAX = 23;
constexpr int NCOLMAX = 11;
/* EoS output columns */
enum { C_T = 0, C_MUB, C_MUS, C_MUQ, C_P, C_CS2, C_E, C_WS, C_WB, C_WSQ, C_WQ };

/* ---------------------------------------------------------------- affine numbers: c + sum_k v[k] X_k ---- */
struct Aff {
  double c;
  double v[NUMAX];
  Aff() : c(0.0) { for (int k = 0; k < NUMAX; ++k) v[k] = 0.0; }
  Aff(double x) : c(x) { for (int k = 0; k < NUMAX; ++k) v[k] = 0.0; }
};
static Aff unknown(int k) { Aff a; a.v[k] = 1.0; return a; }
static Aff operator+(const Aff& a, const Aff& b) { Aff r; r.c = a.c + b.c; for (int k = 0; k < NUMAX; ++k) r.v[k] = a.v[k] + b.v[k]; return r; }
static Aff operator-(const Aff& a, const Aff& b) { Aff r; r.c = a.c - b.c; for (int k = 0; k < NUMAX; ++k) r.v[k] = a.v[k] - b.v[k]; return r; }
static Aff operator-(const Aff& a) { Aff r; r.c = -a.c; for (int k = 0; k < NUMAX; ++k) r.v[k] = -a.v[k]; return r; }
static Aff operator*(double s, const Aff& a) { Aff r; r.c = s * a.c; for (int k = 0; k < NUMAX; ++k) r.v[k] = s * a.v[k]; return r; }
static Aff operator*(const Aff& a, double s) { return s * a; }
static double eval(const Aff& a, const double* x, int nu) { double r = a.c; for (int k = 0; k < nu; ++k) r += a.v[k] * x[k]; return r; }

/* ------------------------------------------------------------------------------------------- containers ---- */
struct State { std::vector<double> f[OF_NSTATE]; };

struct Thermo {
  double T, mu[NQ], p, e, cs2, ws, wq[NQ];
  int oob;
};

struct Derived {
  std::vector<double> sigma_star, s_star, rho_star[NQ], gamma, sigma, s, n[NQ];
  std::vector<Thermo> th;
  std::vector<double> theta, divv, fm[3], fk[NQ];
  std::vector<double> diag[4];       /* Kn_pi, Re_pi^-1, Kn_Pi, Re_Pi^-1 (Eq. 58-61) */
  std::vector<double> fo[9];         /* d_mu eps (4), n_mu (4), |d sigma| (Eq. 145-148) */
  std::vector<double> cell, nnb;
  /* per-particle pair inputs (Step 5): P/sigma*^2, B^j_i/sigma*^2, K^j_q/sigma*^2, alpha_q, v^i */
  std::vector<double> Ppair, Bpair[3][3], Kpair[NQ][3], alpha[NQ], v[3];
  /* gradient sums (Step 4) */
  std::vector<double> FP[3], FB[3], FK[NQ], DU[3][3], DA[NQ][3];
  /* CSR neighbour list (excluding self), indices ascending */
  std::vector<int64_t> nb_off;
  std::vector<int32_t> nb_idx;
  int64_t n_oob = 0;
  int64_t n_oob_steps = 0;   /* summed over the evaluations of rk_step since the last load */
};

struct Table {
  bool loaded = false;
  int32_t dims[4] = {0, 0, 0, 0}, kind[4] = {0, 0, 0, 0}, ncols = 0;
  int32_t col_of[NCOLMAX];
  std::vector<double> ax[4];
  std::vector<double> data;
};

}  // namespace

struct oracle_ctx {
  oracle_params P;
  int64_t N = 0;
  bool loaded = false, derived_valid = false;
  double x0 = 0.0;
  State y;
  State rate;
  Derived d;
  Table tab;
  std::vector<double> src[7];   /* I^0..I^3, I_B, I_S, I_Q per particle (empty: zero), Eq. 38 */
  std::string err;
};

namespace {

/* ---------------------------------------------------------------------------------------------- Step 0 ---- */
struct Geometry {
  double glo[4], gup[4], dglo[4];   /* g_mumu, g^mumu, d g_mumu / dx0 (diagonal metric, mostly minus) */
  double Gam[4][4][4];              /* Christoffel Gamma^nu_{alpha beta}, index order [nu][alpha][beta] */
  double sqrtg, Gamma_g;            /* sqrt(-g), d ln sqrt(-g) / dx0 */
};

static Geometry geometry(const oracle_params& P, double x0) {
  Geometry g;
  std::memset(&g, 0, sizeof(g));
  g.glo[0] = 1.0; g.glo[1] = -1.0; g.glo[2] = -1.0; g.glo[3] = -1.0;
  g.sqrtg = 1.0; g.Gamma_g = 0.0;
  if (P.coords == 1) {            /* hyperbolic (tau, x, y, eta_s): g = diag(1,-1,-1,-tau^2) */
    const double tau = x0;
    g.glo[3] = -(tau * tau);
    g.dglo[3] = -2.0 * tau;
    g.Gam[0][3][3] = tau;
    g.Gam[3][0][3] = 1.0 / tau;
    g.Gam[3][3][0] = 1.0 / tau;
    g.sqrtg = tau;
    g.Gamma_g = 1.0 / tau;
  }
  for (int m = 0; m < 4; ++m) g.gup[m] = 1.0 / g.glo[m];
  return g;
}

static double lorentz_gamma(const Geometry& g, const double u[4]) {
  /* u_mu u^mu = 1 with the mostly-minus metric (DESIGN reading 6) */
  double s = 1.0;
  for (int i = 1; i <= 3; ++i) s += (-g.glo[i]) * u[i] * u[i];
  return std::sqrt(s);
}

/* ------------------------------------------------------------------------------- kernel, Eq. 77 and 79 ---- */
static double sigma_d(int D, double h) {
  const double pi = 3.14159265358979323846;
  if (D == 1) return 2.0 / (3.0 * h);
  if (D == 2) return 10.0 / (7.0 * pi * h * h);
  return 1.0 / (pi * h * h * h);
}

static double kernel_W(int D, double h, double r) {
  const double q = r / h;
  const double sd = sigma_d(D, h);
  if (q <= 1.0) return sd * (1.0 - 1.5 * q * q + 0.75 * q * q * q);
  if (q <= 2.0) return sd * 0.25 * (2.0 - q) * (2.0 - q) * (2.0 - q);
  return 0.0;
}

/* gradient with respect to r_i of W(|r_i - r_j|), dr = r_i - r_j */
static void kernel_gradW(int D, double h, const double dr[3], double out[3]) {
  double r2 = 0.0;
  for (int i = 0; i < D; ++i) r2 += dr[i] * dr[i];
  const double r = std::sqrt(r2);
  out[0] = out[1] = out[2] = 0.0;
  if (r == 0.0) return;
  const double q = r / h;
  const double sd = sigma_d(D, h);
  double f;
  if (q <= 1.0) f = -3.0 * q + 2.25 * q * q;
  else if (q <= 2.0) f = -0.75 * (2.0 - q) * (2.0 - q);
  else return;
  for (int i = 0; i < D; ++i) out[i] = (sd / h) * f * (dr[i] / r);
}

/* ---------------------------------------------------------------------------------------------- Step 1 ---- */
static inline double dist2(int D, const State& y, int64_t a, int64_t b) {
  const double dx = y.f[OF_R1][a] - y.f[OF_R1][b];
  const double dy = y.f[OF_R2][a] - y.f[OF_R2][b];
  double r2 = dx * dx + dy * dy;
  if (D == 3) {
    const double dz = y.f[OF_R3][a] - y.f[OF_R3][b];
    r2 = r2 + dz * dz;
  }
  return r2;
}

static void build_neighbours(const oracle_params& P, const State& y, int64_t N, Derived& d) {
  const int D = P.dim;
  const double twoh = 2.0 * P.h;
  const double cut2 = twoh * twoh;
  d.nb_off.assign(N + 1, 0);
  d.nb_idx.clear();
  d.cell.assign(N, 0.0);
  d.nnb.assign(N, 0.0);

  /* reported cell id (DESIGN reading 9): edge 2h, origin = exact coordinate minimum, product then floor */
  double xmin[3] = {0, 0, 0}, xmax[3] = {0, 0, 0};
  for (int k = 0; k < D; ++k) {
    xmin[k] = xmax[k] = y.f[OF_R1 + k][0];
    for (int64_t a = 1; a < N; ++a) {
      xmin[k] = std::min(xmin[k], y.f[OF_R1 + k][a]);
      xmax[k] = std::max(xmax[k], y.f[OF_R1 + k][a]);
    }
  }
  {
    const double inv_edge = 1.0 / twoh;
    int64_t nc[3] = {1, 1, 1};
    for (int k = 0; k < D; ++k) nc[k] = (int64_t)std::floor((xmax[k] - xmin[k]) * inv_edge) + 1;
    for (int64_t a = 0; a < N; ++a) {
      int64_t c[3] = {0, 0, 0};
      for (int k = 0; k < D; ++k) c[k] = (int64_t)std::floor((y.f[OF_R1 + k][a] - xmin[k]) * inv_edge);
      d.cell[a] = (double)(c[0] + nc[0] * (c[1] + nc[1] * c[2]));
    }
  }

  std::vector<std::vector<int32_t>> lists(N);
  if (P.neighbour_mode == 1) {
    /* O(N^2) definition: b is a neighbour of a iff r_ab^2 < (2h)^2, strictly (DESIGN reading 8) */
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t a = 0; a < N; ++a)
      for (int64_t b = 0; b < N; ++b)
        if (b != a && dist2(D, y, a, b) < cut2) lists[a].push_back((int32_t)b);
  } else {
    /* uniform binning grid (:1434).  The traversal grid is slightly wider than 2h so that rounding in the
       cell index can never hide a pair; the decision itself is the strict r^2 test above. */
    const double edge = twoh * 1.000001;
    const double inv = 1.0 / edge;
    int64_t nc[3] = {1, 1, 1};
    for (int k = 0; k < D; ++k) nc[k] = (int64_t)std::floor((xmax[k] - xmin[k]) * inv) + 1;
    const int64_t ncell = nc[0] * nc[1] * nc[2];
    std::vector<int64_t> cid(N), start(ncell + 1, 0);
    std::vector<int32_t> order(N);
    for (int64_t a = 0; a < N; ++a) {
      int64_t c[3] = {0, 0, 0};
      for (int k = 0; k < D; ++k) c[k] = (int64_t)std::floor((y.f[OF_R1 + k][a] - xmin[k]) * inv);
      cid[a] = c[0] + nc[0] * (c[1] + nc[1] * c[2]);
      start[cid[a] + 1]++;
    }
    for (int64_t c = 0; c < ncell; ++c) start[c + 1] += start[c];
    {
      std::vector<int64_t> fill(start.begin(), start.end() - 1);
      for (int64_t a = 0; a < N; ++a) order[fill[cid[a]]++] = (int32_t)a;
    }
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t a = 0; a < N; ++a) {
      int64_t c[3] = {0, 0, 0};
      int64_t id = cid[a];
      c[0] = id % nc[0]; id /= nc[0]; c[1] = id % nc[1]; c[2] = id / nc[1];
      const int z0 = (D == 3) ? -1 : 0, z1 = (D == 3) ? 1 : 0;
      for (int dz = z0; dz <= z1; ++dz)
        for (int dy = -1; dy <= 1; ++dy)
          for (int dx = -1; dx <= 1; ++dx) {
            const int64_t cx = c[0] + dx, cy = c[1] + dy, cz = c[2] + dz;
            if (cx < 0 || cx >= nc[0] || cy < 0 || cy >= nc[1] || cz < 0 || cz >= nc[2]) continue;
            const int64_t cc = cx + nc[0] * (cy + nc[1] * cz);
            for (int64_t k = start[cc]; k < start[cc + 1]; ++k) {
              const int32_t b = order[k];
              if (b != a && dist2(D, y, a, b) < cut2) lists[a].push_back(b);
            }
          }
      std::sort(lists[a].begin(), lists[a].end());
    }
  }
  for (int64_t a = 0; a < N; ++a) d.nb_off[a + 1] = d.nb_off[a] + (int64_t)lists[a].size();
  d.nb_idx.resize(d.nb_off[N]);
  for (int64_t a = 0; a < N; ++a) {
    std::copy(lists[a].begin(), lists[a].end(), d.nb_idx.begin() + d.nb_off[a]);
    d.nnb[a] = (double)lists[a].size();
  }
}

/* ---------------------------------------------------------------------------------------------- Step 2 ---- */
static void smoothing_sums(const oracle_params& P, const State& y, int64_t N, Derived& d) {
  const int D = P.dim;
  d.sigma_star.assign(N, 0.0);
  d.s_star.assign(N, 0.0);
  for (int q = 0; q < NQ; ++q) d.rho_star[q].assign(N, 0.0);
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t a = 0; a < N; ++a) {
    /* Eq. 72 and Eq. 71 with q*_b / sigma*_b = S_b, N_q,b (Eq. 84-86); b = a is part of the sum */
    const double W0 = kernel_W(D, P.h, 0.0);
    double sg = y.f[OF_MASS][a] * W0;
    double ss = y.f[OF_MASS][a] * y.f[OF_S][a] * W0;
    double rq[NQ];
    for (int q = 0; q < NQ; ++q) rq[q] = y.f[OF_MASS][a] * y.f[OF_NB + q][a] * W0;
    for (int64_t k = d.nb_off[a]; k < d.nb_off[a + 1]; ++k) {
      const int64_t b = d.nb_idx[k];
      const double W = kernel_W(D, P.h, std::sqrt(dist2(D, y, a, b)));
      const double mW = y.f[OF_MASS][b] * W;
      sg += mW;
      ss += mW * y.f[OF_S][b];
      for (int q = 0; q < NQ; ++q) rq[q] += mW * y.f[OF_NB + q][b];
    }
    d.sigma_star[a] = sg;
    d.s_star[a] = ss;
    for (int q = 0; q < NQ; ++q) d.rho_star[q][a] = rq[q];
  }
}

/* ---------------------------------------------------------------------------------------------- Step 3 ---- */
/* forward conformal EoS, an instance of Eq. A.5 (:2115) with A0 = c0, T0 = 1:
   p = c0 T^4 + c2 T^2 sum mu_q^2 + c4 sum mu_q^4;  s = dp/dT, n_q = dp/dmu_q (Eq. A.6-A.7);  e = 3p (:2132) */
static void eos_forward(const oracle_params& P, double T, const double mu[NQ], double& p, double& s, double n[NQ]) {
  double m2 = 0.0, m4 = 0.0;
  for (int q = 0; q < NQ; ++q) { m2 += mu[q] * mu[q]; m4 += mu[q] * mu[q] * mu[q] * mu[q]; }
  p = P.eos_c0 * T * T * T * T + P.eos_c2 * T * T * m2 + P.eos_c4 * m4;
  s = 4.0 * P.eos_c0 * T * T * T + 2.0 * P.eos_c2 * T * m2;
  for (int q = 0; q < NQ; ++q) n[q] = 2.0 * P.eos_c2 * T * T * mu[q] + 4.0 * P.eos_c4 * mu[q] * mu[q] * mu[q];
}

/* single real root of 4 c4 mu^3 + 2 c2 T^2 mu - n = 0, in the closed form of Eq. A.13-A.14 (:2146-2152)
   for chi^3 + alpha1 chi - alpha2 = 0 */
static double mu_of_T(const oracle_params& P, double T, double n) {
  if (n == 0.0) return 0.0;
  if (P.eos_c4 == 0.0) return n / (2.0 * P.eos_c2 * T * T);
  const double sgn = (n < 0.0) ? -1.0 : 1.0;
  const double alpha1 = P.eos_c2 * T * T / (2.0 * P.eos_c4);
  const double alpha2 = std::fabs(n) / (4.0 * P.eos_c4);
  const double delta = std::sqrt(12.0 * alpha1 * alpha1 * alpha1 + 81.0 * alpha2 * alpha2) + 9.0 * alpha2;
  const double d13 = std::cbrt(delta);
  const double chi = (std::cbrt(2.0) * d13 * d13 - 2.0 * std::cbrt(3.0) * alpha1) / (std::cbrt(36.0) * d13);
  return sgn * chi;
}

/* solve of a 4x4 (or n x n) dense system by Gaussian elimination with partial pivoting */
static bool dense_solve(int n, double* A /* n x n row-major */, double* b) {
  for (int c = 0; c < n; ++c) {
    int piv = c;
    for (int r = c + 1; r < n; ++r) if (std::fabs(A[r * n + c]) > std::fabs(A[piv * n + c])) piv = r;
    if (A[piv * n + c] == 0.0) return false;
    if (piv != c) {
      for (int k = 0; k < n; ++k) std::swap(A[c * n + k], A[piv * n + k]);
      std::swap(b[c], b[piv]);
    }
    for (int r = c + 1; r < n; ++r) {
      const double f = A[r * n + c] / A[c * n + c];
      if (f == 0.0) continue;
      for (int k = c; k < n; ++k) A[r * n + k] -= f * A[c * n + k];
      b[r] -= f * b[c];
    }
  }
  for (int r = n - 1; r >= 0; --r) {
    double s = b[r];
    for (int k = r + 1; k < n; ++k) s -= A[r * n + k] * b[k];
    b[r] = s / A[r * n + r];
  }
  return true;
}

/* inversion (s, n_q) -> (T, mu_q): cubic for mu_q(T), then a 1-D monotone solve in T (the analogue of
   Eq. A.15 with s as the key), by bisection to the last bit */
static Thermo eos_closed_form(const oracle_params& P, double s, const double n[NQ]) {
  Thermo th;
  std::memset(&th, 0, sizeof(th));
  double T;
  if (n[0] == 0.0 && n[1] == 0.0 && n[2] == 0.0) {
    T = std::cbrt(s / (4.0 * P.eos_c0));
  } else {
    double lo = 0.0, hi = std::cbrt(s / (4.0 * P.eos_c0));
    for (int it = 0; it < 200; ++it) {
      const double mid = 0.5 * (lo + hi);
      if (mid <= lo || mid >= hi) break;
      double m2 = 0.0;
      for (int q = 0; q < NQ; ++q) { const double m = mu_of_T(P, mid, n[q]); m2 += m * m; }
      const double f = 4.0 * P.eos_c0 * mid * mid * mid + 2.0 * P.eos_c2 * mid * m2 - s;
      if (f > 0.0) hi = mid; else lo = mid;
    }
    T = 0.5 * (lo + hi);
  }
  th.T = T;
  for (int q = 0; q < NQ; ++q) th.mu[q] = mu_of_T(P, T, n[q]);
  double p, s2, n2[NQ];
  eos_forward(P, T, th.mu, p, s2, n2);
  th.p = p;
  th.e = 3.0 * p;
  th.cs2 = 1.0 / 3.0;
  /* w_s = dw/ds|_n, w_q = dw/dn_q|_s from w = T s + sum mu_q n_q and the Jacobian d(T,mu)/d(s,n) = H^-1,
     H = Hessian of p (Eq. A.8-A.10): w_s = T + [H^-1 (s,n)]_0, w_q = mu_q + [H^-1 (s,n)]_q */
  double H[16], z[4];
  std::memset(H, 0, sizeof(H));
  double m2 = 0.0;
  for (int q = 0; q < NQ; ++q) m2 += th.mu[q] * th.mu[q];
  H[0] = 12.0 * P.eos_c0 * T * T + 2.0 * P.eos_c2 * m2;
  for (int q = 0; q < NQ; ++q) {
    H[0 * 4 + (q + 1)] = H[(q + 1) * 4 + 0] = 4.0 * P.eos_c2 * T * th.mu[q];
    H[(q + 1) * 4 + (q + 1)] = 2.0 * P.eos_c2 * T * T + 12.0 * P.eos_c4 * th.mu[q] * th.mu[q];
  }
  z[0] = s; z[1] = n[0]; z[2] = n[1]; z[3] = n[2];
  if (dense_solve(4, H, z)) {
    th.ws = T + z[0];
    for (int q = 0; q < NQ; ++q) th.wq[q] = th.mu[q] + z[q + 1];
  } else {           /* c2 = 0 and mu = 0: charges decouple */
    th.ws = T + T / 3.0;
    for (int q = 0; q < NQ; ++q) th.wq[q] = 0.0;
  }
  th.oob = 0;
  return th;
}

/* offline-inverted table on (s, B, S, Q) axes read by quadrilinear interpolation (:583-593); per axis the
   coordinate is the density itself (kind 0) or its ratio to s (kind 1); out of range: clamp and count */
static Thermo eos_table(const Table& tb, double s, const double n[NQ]) {
  Thermo th;
  std::memset(&th, 0, sizeof(th));
  double x[4];
  x[0] = s;
  for (int k = 1; k < 4; ++k) x[k] = (tb.kind[k] == 1) ? n[k - 1] / s : n[k - 1];
  int i0[4];
  double t[4];
  for (int k = 0; k < 4; ++k) {
    const std::vector<double>& ax = tb.ax[k];
    const int nn = tb.dims[k];
    double xv = x[k];
    if (!(xv >= ax[0])) { xv = ax[0]; th.oob = 1; }
    if (!(xv <= ax[nn - 1])) { xv = ax[nn - 1]; th.oob = 1; }
    int i = (int)(std::upper_bound(ax.begin(), ax.end(), xv) - ax.begin()) - 1;   /* last node <= xv */
    if (i > nn - 2) i = nn - 2;
    if (i < 0) i = 0;
    i0[k] = i;
    t[k] = (xv - ax[i]) / (ax[i + 1] - ax[i]);
  }
  double out[NCOLMAX];
  for (int c = 0; c < NCOLMAX; ++c) out[c] = 0.0;
  for (int b0 = 0; b0 < 2; ++b0)
    for (int b1 = 0; b1 < 2; ++b1)
      for (int b2 = 0; b2 < 2; ++b2)
        for (int b3 = 0; b3 < 2; ++b3) {
          const double w0 = b0 ? t[0] : 1.0 - t[0];
          const double w1 = b1 ? t[1] : 1.0 - t[1];
          const double w2 = b2 ? t[2] : 1.0 - t[2];
          const double w3 = b3 ? t[3] : 1.0 - t[3];
          const double w = ((w0 * w1) * w2) * w3;
          const int64_t node = (((int64_t)(i0[0] + b0) * tb.dims[1] + (i0[1] + b1)) * tb.dims[2] + (i0[2] + b2)) * tb.dims[3] + (i0[3] + b3);
          for (int c = 0; c < NCOLMAX; ++c)
            if (tb.col_of[c] >= 0) out[c] += w * tb.data[node * tb.ncols + tb.col_of[c]];
        }
  th.T = out[C_T];
  for (int q = 0; q < NQ; ++q) { th.mu[q] = out[C_MUB + q]; th.wq[q] = out[C_WB + q]; }
  th.p = out[C_P]; th.cs2 = out[C_CS2]; th.e = out[C_E]; th.ws = out[C_WS];
  return th;
}

/* ------------------------------------------------ offline inverter on a tabulated forward EoS (:576-593) ---- */
/* PAPER.md :583 ("takes a given EoS on a fixed grid of {T, mu} coupled with the backup EoS and then converts this to a
   single EoS table on a fixed grid in {s, n}"), :587 ("the offline inversion procedure uses the existing root-finder and
   interpolator").  The paper prints neither; DESIGN reading 21 fixes them, and this follows it step by step:
     interpolator   quadrilinear blend of the forward columns (p, s, n_B, n_S, n_Q) at X = (T, mu_B, mu_S, mu_Q), X clamped
                    to the grid box; the Jacobian J_ik = d(s, n)_i / dX_k is the derivative of that blend inside its cell
     start          mu_q = 0 (clamped to the axis), T by 60 bisections of s(T, mu) = s* over the T axis
     root-finder    damped Newton, at most 40 iterations: converged when max_i |Y_i - Y*_i| <= 1e-13 s*; J delta = -(Y - Y*)
                    by dense elimination; lambda = 1, 1/2, ... (at most 12 halvings) until the squared residual decreases
     result         T, mu = X; p = blend; e = T s* - p + mu_q n*_q (Euler relation); z = J^-T Y*: dw/ds = T + z_0,
                    dw/dn_q = mu_q + z_q (chain rule on w = T s + mu_q n_q); c_s^2 = (Y* . J^-1 Y*) / (X . Y*), i.e. dp/de
                    along fixed n_q / s (dp = Y . dX, de = X . dY)
     backup EoS     a target the root-finder does not reach (singular J, no decrease, iterations used up) takes the
                    closed-form conformal EoS of the parameters (:572: "progressively moves on to the next EoS"), flag 1 */
struct FwdTable {
  int32_t dims[4];
  const double* ax[4];
  const double* data;      /* [node][5]: p, s, n_B, n_S, n_Q; node = ((i0 * d1 + i1) * d2 + i2) * d3 + i3 */
};

static void fwd_interp(const FwdTable& ft, const double Xin[4], double Y[5], double J[16]) {
  int i0[4];
  double t[4], w[4];
  for (int k = 0; k < 4; ++k) {
    const double* ax = ft.ax[k];
    const int nn = ft.dims[k];
    double xv = Xin[k];
    if (!(xv >= ax[0])) xv = ax[0];
    if (!(xv <= ax[nn - 1])) xv = ax[nn - 1];
    int i = (int)(std::upper_bound(ax, ax + nn, xv) - ax) - 1;
    if (i > nn - 2) i = nn - 2;
    if (i < 0) i = 0;
    i0[k] = i;
    w[k] = ax[i + 1] - ax[i];
    t[k] = (xv - ax[i]) / w[k];
  }
  for (int c = 0; c < 5; ++c) Y[c] = 0.0;
  for (int k = 0; k < 16; ++k) J[k] = 0.0;
  for (int corner = 0; corner < 16; ++corner) {
    int b[4];
    for (int k = 0; k < 4; ++k) b[k] = (corner >> (3 - k)) & 1;
    const int64_t node = (((int64_t)(i0[0] + b[0]) * ft.dims[1] + (i0[1] + b[1])) * ft.dims[2] + (i0[2] + b[2])) * ft.dims[3] + (i0[3] + b[3]);
    const double* f = ft.data + node * 5;
    double wk[4];
    for (int k = 0; k < 4; ++k) wk[k] = b[k] ? t[k] : 1.0 - t[k];
    const double wall = ((wk[0] * wk[1]) * wk[2]) * wk[3];
    for (int c = 0; c < 5; ++c) Y[c] += wall * f[c];
    for (int k = 0; k < 4; ++k) {
      /* d/dX_k of the blend: the weight of axis k is replaced by -+ 1 / (cell width) */
      double wd = (b[k] ? 1.0 : -1.0) / w[k];
      for (int m = 0; m < 4; ++m) if (m != k) wd *= wk[m];
      for (int i = 0; i < 4; ++i) J[i * 4 + k] += wd * f[1 + i];
    }
  }
}

static Thermo invert_forward_point(const oracle_params& P, const FwdTable& ft, double s, const double n[NQ], int32_t& flag,
                                   int32_t& iters) {
  const double Ys[4] = {s, n[0], n[1], n[2]};
  double X[4], Y[5], J[16];
  auto clampX = [&](double* x) {
    for (int k = 0; k < 4; ++k) {
      if (!(x[k] >= ft.ax[k][0])) x[k] = ft.ax[k][0];
      if (!(x[k] <= ft.ax[k][ft.dims[k] - 1])) x[k] = ft.ax[k][ft.dims[k] - 1];
    }
  };
  auto res2 = [&](const double* y) {
    double r = 0.0;
    for (int i = 0; i < 4; ++i) { const double d = (y[1 + i] - Ys[i]) / s; r += d * d; }
    return r;
  };
  /* start */
  X[0] = 0.0; X[1] = X[2] = X[3] = 0.0;
  clampX(X);
  {
    double lo = ft.ax[0][0], hi = ft.ax[0][ft.dims[0] - 1];
    for (int it = 0; it < 60; ++it) {
      const double mid = 0.5 * (lo + hi);
      X[0] = mid;
      fwd_interp(ft, X, Y, J);
      if (Y[1] > s) hi = mid; else lo = mid;
    }
    X[0] = 0.5 * (lo + hi);
  }
  fwd_interp(ft, X, Y, J);
  bool ok = false;
  iters = 0;
  for (int it = 0; it < 40; ++it) {
    double rmax = 0.0;
    for (int i = 0; i < 4; ++i) rmax = std::max(rmax, std::fabs(Y[1 + i] - Ys[i]));
    if (rmax <= 1e-13 * s) { ok = true; break; }
    double A[16], d[4];
    for (int k = 0; k < 16; ++k) A[k] = J[k];
    for (int i = 0; i < 4; ++i) d[i] = -(Y[1 + i] - Ys[i]);
    if (!dense_solve(4, A, d)) break;
    const double r0 = res2(Y);
    double lam = 1.0;
    bool acc = false;
    for (int hv = 0; hv <= 12; ++hv) {
      double Xn[4], Yn[5], Jn[16];
      for (int k = 0; k < 4; ++k) Xn[k] = X[k] + lam * d[k];
      clampX(Xn);
      fwd_interp(ft, Xn, Yn, Jn);
      if (res2(Yn) < r0) {
        for (int k = 0; k < 4; ++k) X[k] = Xn[k];
        for (int c = 0; c < 5; ++c) Y[c] = Yn[c];
        for (int k = 0; k < 16; ++k) J[k] = Jn[k];
        acc = true;
        break;
      }
      lam *= 0.5;
    }
    ++iters;
    if (!acc) break;
  }
  if (!ok) {
    double rmax = 0.0;
    for (int i = 0; i < 4; ++i) rmax = std::max(rmax, std::fabs(Y[1 + i] - Ys[i]));
    ok = rmax <= 1e-13 * s;
  }
  Thermo th;
  std::memset(&th, 0, sizeof(th));
  double A[16], z[4], v[4];
  if (ok) {
    for (int i = 0; i < 4; ++i) for (int k = 0; k < 4; ++k) A[i * 4 + k] = J[k * 4 + i];     /* J^T */
    for (int i = 0; i < 4; ++i) z[i] = Ys[i];
    ok = dense_solve(4, A, z);
  }
  if (ok) {
    for (int k = 0; k < 16; ++k) A[k] = J[k];
    for (int i = 0; i < 4; ++i) v[i] = Ys[i];
    ok = dense_solve(4, A, v);
  }
  if (!ok) {
    flag = 1;
    return eos_closed_form(P, s, n);
  }
  flag = 0;
  th.T = X[0];
  for (int q = 0; q < NQ; ++q) th.mu[q] = X[1 + q];
  th.p = Y[0];
  th.e = X[0] * s - Y[0] + (X[1] * n[0] + X[2] * n[1] + X[3] * n[2]);
  th.ws = X[0] + z[0];
  for (int q = 0; q < NQ; ++q) th.wq[q] = X[1 + q] + z[1 + q];
  double num = 0.0, den = 0.0;
  for (int i = 0; i < 4; ++i) { num += Ys[i] * v[i]; den += X[i] * Ys[i]; }
  th.cs2 = num / den;
  return th;
}

/* transport coefficients, §5.3 :732-769 and DESIGN reading 11 */
struct Transport { double eta, zeta, tau_pi, tau_Pi, kappa[NQ][NQ], tau_q[NQ]; };

static Transport transport(const oracle_params& P, const Thermo& th, double s) {
  Transport tr;
  const double w = th.e + th.p;
  tr.eta = P.eta_over_s * s;                                      /* constant eta/s (:734) */
  tr.tau_pi = std::max(P.tau_pi_coeff * tr.eta / w, P.tau_floor);
  const double dT = th.T - P.zeta_T_peak;
  tr.zeta = (P.zeta_width > 0.0)
                ? P.zeta_max * (P.zeta_width * P.zeta_width) / (P.zeta_width * P.zeta_width + dT * dT) * s
                : P.zeta_max * s;                                 /* constant zeta/s (:756) */
  tr.tau_Pi = P.tau_Pi_coeff * tr.tau_pi;
  for (int q = 0; q < NQ; ++q) {
    for (int r = 0; r < NQ; ++r) tr.kappa[q][r] = P.kappa_over_T2[q * 3 + r] * th.T * th.T;  /* :769, :779 */
    tr.tau_q[q] = P.tau_q_times_T[q] / th.T;                                              /* :781 */
  }
  return tr;
}

/* reconstructed dissipative tensors of one particle (Step 6: time components from u_mu pi^{mu nu} = 0,
   u_mu J^mu = 0, never evolved) */
struct Dissip {
  double pit[4][4];     /* pi~^{mu nu} = pi^{mu nu} / sigma */
  double Jt[NQ][4];     /* J~^mu_q */
  double bulkt;         /* Pi~ */
};

static bool shear_on(const oracle_params& P) { return P.eom != 0 && (P.flags & 1); }
static bool bulk_on(const oracle_params& P) { return P.eom != 0 && (P.flags & 2); }
static bool diff_on(const oracle_params& P) { return P.eom != 0 && (P.flags & 4); }

static Dissip dissipative(const oracle_params& P, const Geometry& g, const State& y, int64_t a, const double u[4]) {
  Dissip ds;
  std::memset(&ds, 0, sizeof(ds));
  const int D = P.dim;
  const double gam = u[0];
  if (bulk_on(P)) ds.bulkt = y.f[OF_BULK][a];
  if (shear_on(P)) {
    ds.pit[1][1] = y.f[OF_PI11][a];
    ds.pit[1][2] = ds.pit[2][1] = y.f[OF_PI12][a];
    ds.pit[2][2] = y.f[OF_PI22][a];
    ds.pit[3][3] = y.f[OF_PI33][a];
    if (D == 3) {
      ds.pit[1][3] = ds.pit[3][1] = y.f[OF_PI13][a];
      ds.pit[2][3] = ds.pit[3][2] = y.f[OF_PI23][a];
    }
    /* u_mu pi^{mu i} = 0  =>  gamma pi^{0 i} = sum_j G_j u^j pi^{j i};  then pi^{00} from pi^{j0} */
    for (int i = 1; i <= 3; ++i) {
      double sacc = 0.0;
      for (int j = 1; j <= 3; ++j) sacc += (-g.glo[j]) * u[j] * ds.pit[j][i];
      ds.pit[0][i] = ds.pit[i][0] = sacc / gam;
    }
    double sacc = 0.0;
    for (int j = 1; j <= 3; ++j) sacc += (-g.glo[j]) * u[j] * ds.pit[j][0];
    ds.pit[0][0] = sacc / gam;
  }
  if (diff_on(P)) {
    for (int q = 0; q < NQ; ++q) {
      for (int i = 1; i <= D; ++i) ds.Jt[q][i] = y.f[OF_JB1 + 3 * q + (i - 1)][a];
      double sacc = 0.0;
      for (int j = 1; j <= 3; ++j) sacc += (-g.glo[j]) * u[j] * ds.Jt[q][j];
      ds.Jt[q][0] = sacc / gam;
    }
  }
  return ds;
}

static void four_velocity(const oracle_params& P, const Geometry& g, const State& y, int64_t a, double u[4]) {
  u[1] = y.f[OF_U1][a];
  u[2] = y.f[OF_U2][a];
  u[3] = (P.dim == 3) ? y.f[OF_U3][a] : 0.0;
  u[0] = 0.0;
  u[0] = lorentz_gamma(g, u);
}

static void thermo_pass(oracle_ctx* c, const State& y, double x0, Derived& d) {
  const oracle_params& P = c->P;
  const int64_t N = c->N;
  const int D = P.dim;
  const Geometry g = geometry(P, x0);
  d.gamma.assign(N, 0.0); d.sigma.assign(N, 0.0); d.s.assign(N, 0.0);
  for (int q = 0; q < NQ; ++q) { d.n[q].assign(N, 0.0); d.alpha[q].assign(N, 0.0); d.FK[q].assign(N, 0.0); }
  d.th.assign(N, Thermo());
  d.Ppair.assign(N, 0.0);
  for (int j = 0; j < 3; ++j) {
    d.v[j].assign(N, 0.0);
    for (int i = 0; i < 3; ++i) d.Bpair[j][i].assign(N, 0.0);
    for (int q = 0; q < NQ; ++q) d.Kpair[q][j].assign(N, 0.0);
  }
  int64_t n_oob = 0;
#pragma omp parallel for schedule(dynamic, 64) reduction(+ : n_oob)
  for (int64_t a = 0; a < N; ++a) {
    double u[4];
    four_velocity(P, g, y, a, u);
    const double gam = u[0];
    d.gamma[a] = gam;
    /* Eq. 68: rest-frame density = lab-frame density / (u^0 sqrt(-g)) (DESIGN reading 2) */
    const double lab = gam * g.sqrtg;
    d.sigma[a] = d.sigma_star[a] / lab;
    d.s[a] = d.s_star[a] / lab;
    double n[NQ];
    for (int q = 0; q < NQ; ++q) { n[q] = d.rho_star[q][a] / lab; d.n[q][a] = n[q]; }
    Thermo th = (P.eos_kind == 0) ? eos_closed_form(P, d.s[a], n) : eos_table(c->tab, d.s[a], n);
    n_oob += th.oob;
    d.th[a] = th;
    const double sig = d.sigma[a], sst2 = d.sigma_star[a] * d.sigma_star[a];
    const Dissip ds = dissipative(P, g, y, a, u);
    for (int j = 1; j <= D; ++j) d.v[j - 1][a] = u[j] / gam;
    for (int q = 0; q < NQ; ++q) d.alpha[q][a] = th.mu[q] / th.T;
    /* pair inputs of Step 5: (p + Pi), B^j_i = pi^j_i - v^j pi^0_i, K^j_q = J^j_q - v^j J^0_q, each / sigma*^2 */
    d.Ppair[a] = (th.p + ds.bulkt * sig) / sst2;
    for (int j = 1; j <= D; ++j)
      for (int i = 1; i <= D; ++i) {
        const double pi_j_i = sig * ds.pit[j][i] * g.glo[i];
        const double pi_0_i = sig * ds.pit[0][i] * g.glo[i];
        d.Bpair[j - 1][i - 1][a] = (pi_j_i - (u[j] / gam) * pi_0_i) / sst2;
      }
    for (int q = 0; q < NQ; ++q)
      for (int j = 1; j <= D; ++j)
        d.Kpair[q][j - 1][a] = (sig * ds.Jt[q][j] - (u[j] / gam) * sig * ds.Jt[q][0]) / sst2;
  }
  d.n_oob = n_oob;
}

/* ---------------------------------------------------------------------------------------------- Step 4 ---- */
static void gradient_sums(const oracle_params& P, const State& y, int64_t N, Derived& d) {
  const int D = P.dim;
  for (int i = 0; i < 3; ++i) {
    d.FP[i].assign(N, 0.0); d.FB[i].assign(N, 0.0);
    for (int j = 0; j < 3; ++j) d.DU[j][i].assign(N, 0.0);
    for (int q = 0; q < NQ; ++q) d.DA[q][i].assign(N, 0.0);
  }
  for (int q = 0; q < NQ; ++q) d.FK[q].assign(N, 0.0);
  d.divv.assign(N, 0.0);
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t a = 0; a < N; ++a) {
    double FP[3] = {0, 0, 0}, FB[3] = {0, 0, 0}, FK[NQ] = {0, 0, 0}, DU[3][3] = {{0}}, DA[NQ][3] = {{0}}, dv = 0.0;
    for (int64_t k = d.nb_off[a]; k < d.nb_off[a + 1]; ++k) {
      const int64_t b = d.nb_idx[k];
      double dr[3] = {0, 0, 0}, gW[3];
      for (int i = 0; i < D; ++i) dr[i] = y.f[OF_R1 + i][a] - y.f[OF_R1 + i][b];
      kernel_gradW(D, P.h, dr, gW);                       /* Eq. 79, d_i W_ab */
      const double mb = y.f[OF_MASS][b];
      for (int i = 0; i < D; ++i) {
        /* n = -1 form (pair antisymmetric, :944): (1/sigma*) d_i A = sum m_b [A_a/sigma*_a^2 + A_b/sigma*_b^2] d_i W */
        FP[i] += mb * (d.Ppair[a] + d.Ppair[b]) * gW[i];
        for (int j = 0; j < D; ++j) FB[i] += mb * (d.Bpair[j][i][a] + d.Bpair[j][i][b]) * gW[j];
        /* n = +1 form (pair symmetric): d_j A = (1/sigma*_a) sum m_b (A_b - A_a) d_j W */
        for (int j = 0; j < D; ++j) DU[j][i] += mb * (y.f[OF_U1 + i][b] - y.f[OF_U1 + i][a]) * gW[j];
        dv += mb * (d.v[i][b] - d.v[i][a]) * gW[i];
        for (int q = 0; q < NQ; ++q) DA[q][i] += mb * (d.alpha[q][b] - d.alpha[q][a]) * gW[i];
      }
      for (int q = 0; q < NQ; ++q)
        for (int j = 0; j < D; ++j) FK[q] += mb * (d.Kpair[q][j][a] + d.Kpair[q][j][b]) * gW[j];
    }
    const double inv = 1.0 / d.sigma_star[a];
    for (int i = 0; i < 3; ++i) {
      d.FP[i][a] = FP[i]; d.FB[i][a] = FB[i];
      for (int j = 0; j < 3; ++j) d.DU[j][i][a] = DU[j][i] * inv;
      for (int q = 0; q < NQ; ++q) d.DA[q][i][a] = DA[q][i] * inv;
    }
    for (int q = 0; q < NQ; ++q) d.FK[q][a] = FK[q];
    d.divv[a] = dv * inv;
  }
}

/* ---------------------------------------------------------------------------------------------- Step 5 ---- */
struct Unknowns {
  int D, npi, nu;
  int iu[4];          /* du^i/dx0, i = 1..D  */
  int iS, iN[NQ], iBulk;
  int ipi[4][4];      /* evolved spatial pi~^{ij}; -1 where not evolved */
  int iJ[NQ][4];
};

static Unknowns unknown_layout(int D) {
  Unknowns U;
  U.D = D;
  int k = 0;
  for (int i = 0; i < 4; ++i) U.iu[i] = -1;
  for (int i = 1; i <= D; ++i) U.iu[i] = k++;
  U.iS = k++;
  for (int q = 0; q < NQ; ++q) U.iN[q] = k++;
  U.iBulk = k++;
  for (int i = 0; i < 4; ++i) for (int j = 0; j < 4; ++j) U.ipi[i][j] = -1;
  if (D == 3) {
    const int comp[6][2] = {{1, 1}, {1, 2}, {1, 3}, {2, 2}, {2, 3}, {3, 3}};
    for (auto& c : comp) { U.ipi[c[0]][c[1]] = U.ipi[c[1]][c[0]] = k++; }
    U.npi = 6;
  } else {
    const int comp[4][2] = {{1, 1}, {1, 2}, {2, 2}, {3, 3}};
    for (auto& c : comp) { U.ipi[c[0]][c[1]] = U.ipi[c[1]][c[0]] = k++; }
    U.npi = 4;
  }
  for (int q = 0; q < NQ; ++q) {
    for (int i = 0; i < 4; ++i) U.iJ[q][i] = -1;
    for (int i = 1; i <= D; ++i) U.iJ[q][i] = k++;
  }
  U.nu = k;
  return U;
}

static int state_id_of_pi(int i, int j) {
  if (i > j) std::swap(i, j);
  if (i == 1 && j == 1) return OF_PI11;
  if (i == 1 && j == 2) return OF_PI12;
  if (i == 1 && j == 3) return OF_PI13;
  if (i == 2 && j == 2) return OF_PI22;
  if (i == 2 && j == 3) return OF_PI23;
  return OF_PI33;
}

/* Assemble and solve the linear system of one particle; write the time derivatives into k.
   Returns false on a singular system. */
static bool eom_particle(const oracle_params& P, const Geometry& g, const State& y, const Derived& d, int64_t a,
                         double x0, State& k, double& theta_out, double diag_out[4], const double Isrc[7]) {
  const int D = P.dim;
  const Unknowns U = unknown_layout(D);
  const int NU = U.nu;
  const bool shear = shear_on(P), bulk = bulk_on(P), diff = diff_on(P);

  /* four-velocity and its time derivative */
  double u[4], ulo[4], v[4];
  four_velocity(P, g, y, a, u);
  const double gam = u[0];
  for (int m = 0; m < 4; ++m) { ulo[m] = g.glo[m] * u[m]; v[m] = u[m] / gam; }
  Aff du[4];
  for (int i = 1; i <= D; ++i) du[i] = unknown(U.iu[i]);
  {
    /* Eq. 97 (:1011), nu = 0 component: du^0 = -(u_k/u_0) du^k - u^a u^b (dg_ab/dx0) / (2 u_0) */
    Aff s(0.0);
    for (int kk = 1; kk <= 3; ++kk) s = s - (ulo[kk] / ulo[0]) * du[kk];
    double gt = 0.0;
    for (int m = 0; m < 4; ++m) gt += u[m] * u[m] * g.dglo[m];
    du[0] = s - Aff(gt / (2.0 * ulo[0]));
  }
  Aff dulo[4];
  for (int m = 0; m < 4; ++m) dulo[m] = g.glo[m] * du[m] + Aff(g.dglo[m] * u[m]);

  /* partial derivatives d_mu u^nu: spatial ones from the SPH sums, d_k u^0 from u_mu d_k u^mu = 0,
     d_0 = d/dx0 - v^k d_k (Notation, :167) */
  Aff PU[4][4];
  for (int kk = 1; kk <= D; ++kk) {
    double s0 = 0.0;
    for (int j = 1; j <= D; ++j) {
      PU[kk][j] = Aff(d.DU[kk - 1][j - 1][a]);
      s0 += (-g.glo[j]) * u[j] * d.DU[kk - 1][j - 1][a];
    }
    PU[kk][0] = Aff(s0 / gam);
  }
  for (int n = 0; n < 4; ++n) {
    Aff s = du[n];
    for (int kk = 1; kk <= 3; ++kk) s = s - v[kk] * PU[kk][n];
    PU[0][n] = s;
  }
  /* covariant derivative nabla_mu u^nu = d_mu u^nu + Gamma^nu_{mu lam} u^lam */
  Aff CD[4][4];
  for (int m = 0; m < 4; ++m)
    for (int n = 0; n < 4; ++n) {
      Aff s = PU[m][n];
      for (int l = 0; l < 4; ++l) if (g.Gam[n][m][l] != 0.0) s = s + Aff(g.Gam[n][m][l] * u[l]);
      CD[m][n] = s;
    }
  /* expansion rate (DESIGN reading: theta = gamma [ (div v)_SPH + Gamma_g ] + d gamma / dx0) */
  const Aff theta = Aff(gam * (d.divv[a] + g.Gamma_g)) + du[0];
  /* D u^nu = u^mu nabla_mu u^nu */
  Aff Du[4], Dulo[4];
  for (int n = 0; n < 4; ++n) {
    Aff s(0.0);
    for (int m = 0; m < 4; ++m) s = s + u[m] * CD[m][n];
    Du[n] = s;
    Dulo[n] = g.glo[n] * s;
  }

  /* thermodynamics and transport */
  const Thermo& th = d.th[a];
  const double sig = d.sigma[a];
  const double w = th.e + th.p;
  const Transport tr = transport(P, th, d.s[a]);
  const Dissip ds = dissipative(P, g, y, a, u);
  const double Pi = ds.bulkt * sig;

  /* unknown time derivatives of the evolved variables */
  const Aff dS = unknown(U.iS);
  Aff dN[NQ];
  for (int q = 0; q < NQ; ++q) dN[q] = unknown(U.iN[q]);
  const Aff dBulk = unknown(U.iBulk);
  Aff dpit[4][4];
  for (int i = 1; i <= 3; ++i)
    for (int j = 1; j <= 3; ++j)
      if (U.ipi[i][j] >= 0) dpit[i][j] = unknown(U.ipi[i][j]);
  /* d/dx0 of u_mu pi~^{mu nu} = 0:  gamma dpi~^{0 nu} = - sum_mu du_mu pi~^{mu nu} - sum_j u_j dpi~^{j nu} */
  for (int n = 1; n <= 3; ++n) {
    Aff s(0.0);
    for (int m = 0; m < 4; ++m) s = s - dulo[m] * ds.pit[m][n];
    for (int j = 1; j <= 3; ++j) s = s - ulo[j] * dpit[j][n];
    dpit[0][n] = (1.0 / gam) * s;
    dpit[n][0] = dpit[0][n];
  }
  {
    Aff s(0.0);
    for (int m = 0; m < 4; ++m) s = s - dulo[m] * ds.pit[m][0];
    for (int j = 1; j <= 3; ++j) s = s - ulo[j] * dpit[j][0];
    dpit[0][0] = (1.0 / gam) * s;
  }
  Aff dJt[NQ][4];
  for (int q = 0; q < NQ; ++q) {
    for (int i = 1; i <= D; ++i) dJt[q][i] = unknown(U.iJ[q][i]);
    Aff s(0.0);
    for (int m = 0; m < 4; ++m) s = s - dulo[m] * ds.Jt[q][m];
    for (int j = 1; j <= 3; ++j) s = s - ulo[j] * dJt[q][j];
    dJt[q][0] = (1.0 / gam) * s;
  }

  /* velocity-shear and vorticity tensors, full 4x4 (Notation :169):
     sigma^{mn} = 1/2 (nabla^m u^n + nabla^n u^m) - 1/2 (u^m Du^n + u^n Du^m) - 1/3 Delta^{mn} theta
     omega^{mn} = 1/2 (nabla^m u^n - nabla^n u^m) - 1/2 (u^m Du^n - u^n Du^m)                          */
  Aff sg[4][4], om[4][4];
  {   /* always: the diagnostics of Eq. 58 need sigma^{mn} also for an ideal fluid */
    for (int m = 0; m < 4; ++m)
      for (int n = 0; n < 4; ++n) {
        const Aff up_mn = g.gup[m] * CD[m][n], up_nm = g.gup[n] * CD[n][m];
        const double Delta = ((m == n) ? g.gup[m] : 0.0) - u[m] * u[n];
        sg[m][n] = 0.5 * (up_mn + up_nm) - 0.5 * (u[m] * Du[n] + u[n] * Du[m]) - (Delta / 3.0) * theta;
        om[m][n] = 0.5 * (up_mn - up_nm) - 0.5 * (u[m] * Du[n] - u[n] * Du[m]);
      }
  }

  /* second-order coefficients: minimal IS (Eq. 49-50) is delta_PiPi = tau_Pi, delta_pipi = 4/3 tau_pi, rest 0 */
  double delta_PiPi = tr.tau_Pi, lambda_Pipi = 0.0, delta_pipi = (4.0 / 3.0) * tr.tau_pi, tau_pipi = 0.0,
         lambda_piPi = 0.0, phi_omega = 0.0;
  if (P.eom == 2) {
    delta_PiPi = P.dnmr_coeffs[0] * tr.tau_Pi;
    lambda_Pipi = P.dnmr_coeffs[1] * tr.tau_Pi;
    delta_pipi = P.dnmr_coeffs[2] * tr.tau_pi;
    tau_pipi = P.dnmr_coeffs[3] * tr.tau_pi;
    lambda_piPi = P.dnmr_coeffs[4];
    phi_omega = P.dnmr_coeffs[5];
  }

  /* ---- the equations, each as an affine expression that must vanish ---- */
  std::vector<Aff> eq;
  eq.reserve(NU);

  /* momentum, i = 1..D:  d/dx0 [ C u_i + pi~^0_i / gamma ] = sqrt(-g) ( FP_i - FB_i ),  C = (w + Pi)/sigma */
  const double A = w * th.cs2;
  const double Cc = w / sig + ds.bulkt;
  Aff dC = th.ws * dS + dBulk - (A / sig) * ((1.0 / gam) * theta);
  for (int q = 0; q < NQ; ++q) dC = dC + th.wq[q] * dN[q];
  for (int i = 1; i <= D; ++i) {
    const double pit0_lo = g.glo[i] * ds.pit[0][i];
    const Aff dpit0_lo = Aff(g.dglo[i] * ds.pit[0][i]) + g.glo[i] * dpit[0][i];
    const Aff lhs = ulo[i] * dC + Cc * dulo[i] + (1.0 / gam) * dpit0_lo - (pit0_lo / (gam * gam)) * du[0];
    /* source, Eq. 38 / 43: + sqrt(-g) I_i / sigma* = I_i / (gamma sigma), I_i = g_ii I^i */
    eq.push_back(lhs - Aff(g.sqrtg * (d.FP[i - 1][a] - d.FB[i - 1][a]) + g.glo[i] * Isrc[i] / (gam * sig)));
  }
  /* entropy, Eq. 96 (:1003) with I = 0:  u^0 sigma T dS + u^0 sigma mu_q dN_q = -Pi theta + pi^mu_nu nabla_mu u^nu */
  {
    Aff lhs = (gam * sig * th.T) * dS;
    for (int q = 0; q < NQ; ++q) lhs = lhs + (gam * sig * th.mu[q]) * dN[q];
    Aff rhs = -(Pi * theta);
    for (int m = 0; m < 4; ++m)
      for (int n = 0; n < 4; ++n) {
        const double pi_m_n = sig * ds.pit[m][n] * g.glo[n];
        if (pi_m_n != 0.0) rhs = rhs + pi_m_n * CD[m][n];
      }
    double uI = 0.0;                          /* u_mu I^mu, Eq. 96 */
    for (int m = 0; m < 4; ++m) uI += ulo[m] * Isrc[m];
    rhs = rhs + Aff(uI);
    eq.push_back(lhs - rhs);
  }
  /* charge:  d/dx0 [ N_q + J~^0_q / gamma ] = - sqrt(-g) FK_q */
  for (int q = 0; q < NQ; ++q) {
    const Aff lhs = dN[q] + (1.0 / gam) * dJt[q][0] - (ds.Jt[q][0] / (gam * gam)) * du[0];
    eq.push_back(lhs + Aff(g.sqrtg * d.FK[q][a] - Isrc[4 + q] / (gam * sig)));     /* Eq. 44: + I_q */
  }
  /* bulk (Eq. 49 / Eq. 52 row 1 in terms of Pi~ = Pi/sigma, D sigma = -sigma theta):
     tau_Pi sigma gamma dPi~ = -Pi - zeta theta + (tau_Pi - delta_PiPi) Pi theta + lambda_Pipi pi^{mn} sigma_{mn} */
  if (bulk) {
    Aff rhs = Aff(-Pi) - tr.zeta * theta + ((tr.tau_Pi - delta_PiPi) * Pi) * theta;
    if (lambda_Pipi != 0.0)
      for (int m = 0; m < 4; ++m)
        for (int n = 0; n < 4; ++n) {
          const double pimn = sig * ds.pit[m][n];
          if (pimn != 0.0) rhs = rhs + (lambda_Pipi * pimn * g.glo[m] * g.glo[n]) * sg[m][n];
        }
    eq.push_back((tr.tau_Pi * sig * gam) * dBulk - rhs);
  } else {
    eq.push_back(dBulk);
  }
  /* shear (Eq. 50 / Eq. 52 row 3), evolved components ij:
     sigma tau_pi [ D pi~^{ij} + (u^i pi~^{j l} + u^j pi~^{i l}) Du_l ] =
        -pi^{ij} + 2 eta sigma^{ij} + (tau_pi - delta_pipi) pi^{ij} theta - tau_pipi pi^{l<i} sigma^{j>}_l
        + lambda_piPi Pi sigma^{ij} + 2 tau_pi phi_omega pi^{<i}_l omega^{j>l}                             */
  {
    Aff Xtr(0.0);               /* pi^{l a} sigma_{a l} */
    if (shear && tau_pipi != 0.0)
      for (int l = 0; l < 4; ++l)
        for (int m = 0; m < 4; ++m) {
          const double pilm = sig * ds.pit[l][m];
          if (pilm != 0.0) Xtr = Xtr + (pilm * g.glo[l] * g.glo[m]) * sg[m][l];
        }
    for (int i = 1; i <= 3; ++i)
      for (int j = i; j <= 3; ++j) {
        if (U.ipi[i][j] < 0) continue;
        if (!shear) { eq.push_back(dpit[i][j]); continue; }
        Aff lhs = gam * dpit[i][j];
        for (int l = 0; l < 4; ++l)
          for (int r = 0; r < 4; ++r) {
            if (g.Gam[i][l][r] != 0.0) lhs = lhs + Aff(u[l] * g.Gam[i][l][r] * ds.pit[r][j]);
            if (g.Gam[j][l][r] != 0.0) lhs = lhs + Aff(u[l] * g.Gam[j][l][r] * ds.pit[i][r]);
          }
        for (int l = 0; l < 4; ++l) lhs = lhs + (u[i] * ds.pit[j][l] + u[j] * ds.pit[i][l]) * Dulo[l];
        const double piij = sig * ds.pit[i][j];
        Aff rhs = Aff(-piij) + (2.0 * tr.eta) * sg[i][j] + ((tr.tau_pi - delta_pipi) * piij) * theta;
        if (tau_pipi != 0.0) {
          /* X^{ij} = pi^{l i} sigma^j_l;  X^{<ij>} = 1/2 (X^{ij} + X^{ji}) - 1/3 Delta^{ij} X^a_a */
          Aff X(0.0);
          for (int l = 0; l < 4; ++l) {
            X = X + (0.5 * sig * ds.pit[l][i] * g.glo[l]) * sg[l][j];
            X = X + (0.5 * sig * ds.pit[l][j] * g.glo[l]) * sg[l][i];
          }
          const double Delta = ((i == j) ? g.gup[i] : 0.0) - u[i] * u[j];
          X = X - (Delta / 3.0) * Xtr;
          rhs = rhs - tau_pipi * X;
        }
        if (lambda_piPi != 0.0) rhs = rhs + (lambda_piPi * Pi) * sg[i][j];
        if (phi_omega != 0.0) {
          /* Y^{ij} = pi^i_l omega^{j l}; trace pi^{al} omega_{al} = 0 (symmetric x antisymmetric) */
          Aff Y(0.0);
          for (int l = 0; l < 4; ++l) {
            Y = Y + (0.5 * sig * ds.pit[i][l] * g.glo[l]) * om[j][l];
            Y = Y + (0.5 * sig * ds.pit[j][l] * g.glo[l]) * om[i][l];
          }
          rhs = rhs + (2.0 * tr.tau_pi * phi_omega) * Y;
        }
        eq.push_back((sig * tr.tau_pi) * lhs - rhs);
      }
  }
  /* diffusion (Eq. 51, DESIGN reading 12), diagonal relaxation times:
     tau_q sigma [ D J~^i_q + u^i J~^nu_q Du_nu ] = -J^i_q + sum_q' kappa_qq' nabla^<i> alpha_q',
     nabla^<i> alpha = -(1/G_i) d_i alpha - u^i u^j d_j alpha (the d_0 alpha part is dropped)            */
  for (int q = 0; q < NQ; ++q)
    for (int i = 1; i <= D; ++i) {
      if (!diff) { eq.push_back(dJt[q][i]); continue; }
      Aff lhs = gam * dJt[q][i];
      for (int l = 0; l < 4; ++l)
        for (int r = 0; r < 4; ++r)
          if (g.Gam[i][l][r] != 0.0) lhs = lhs + Aff(u[l] * g.Gam[i][l][r] * ds.Jt[q][r]);
      Aff JDu(0.0);
      for (int n = 0; n < 4; ++n) JDu = JDu + ds.Jt[q][n] * Dulo[n];
      lhs = lhs + u[i] * JDu;
      double rhs = -sig * ds.Jt[q][i];
      for (int r = 0; r < NQ; ++r) {
        double udota = 0.0;
        for (int j = 1; j <= D; ++j) udota += u[j] * d.DA[r][j - 1][a];
        const double proj = g.gup[i] * d.DA[r][i - 1][a] - u[i] * udota;
        rhs += tr.kappa[q][r] * proj;
      }
      eq.push_back((tr.tau_q[q] * sig) * lhs - Aff(rhs));
    }

  if ((int)eq.size() != NU) return false;
  /* dense solve: sum_k eq[r].v[k] X_k = -eq[r].c */
  std::vector<double> M((size_t)NU * NU), rhs(NU);
  for (int r = 0; r < NU; ++r) {
    for (int kk = 0; kk < NU; ++kk) M[(size_t)r * NU + kk] = eq[r].v[kk];
    rhs[r] = -eq[r].c;
  }
  if (!dense_solve(NU, M.data(), rhs.data())) return false;
  const double* X = rhs.data();

  /* derivatives of the evolved set (Step 6) */
  for (int f = 0; f < OF_NSTATE; ++f) k.f[f][a] = 0.0;
  for (int i = 1; i <= D; ++i) {
    k.f[OF_R1 + i - 1][a] = u[i] / gam;          /* dr^i/dx0 = v^i */
    k.f[OF_U1 + i - 1][a] = X[U.iu[i]];
  }
  k.f[OF_S][a] = X[U.iS];
  for (int q = 0; q < NQ; ++q) k.f[OF_NB + q][a] = X[U.iN[q]];
  k.f[OF_BULK][a] = X[U.iBulk];
  for (int i = 1; i <= 3; ++i)
    for (int j = i; j <= 3; ++j)
      if (U.ipi[i][j] >= 0) k.f[state_id_of_pi(i, j)][a] = X[U.ipi[i][j]];
  for (int q = 0; q < NQ; ++q)
    for (int i = 1; i <= D; ++i) k.f[OF_JB1 + 3 * q + i - 1][a] = X[U.iJ[q][i]];
  /* 2+1D hyperbolic: longitudinal work rate per particle (DESIGN reading 14),
     d work / d tau = (m / sigma*) (p + Pi + tau^2 pi^{eta eta}) */
  if (P.coords == 1 && D == 2)
    k.f[OF_WORK][a] = (y.f[OF_MASS][a] / d.sigma_star[a]) * (th.p + Pi + x0 * x0 * sig * ds.pit[3][3]);
  theta_out = eval(theta, X, NU);
  /* applicability diagnostics at the solution, Eq. 58-61 (:797-805); the metric is diagonal, so
     A^{mn} A_{mn} = sum_mn g_mm g_nn (A^{mn})^2 */
  {
    double ss = 0.0, pp = 0.0;
    for (int m = 0; m < 4; ++m)
      for (int n = 0; n < 4; ++n) {
        const double sv = eval(sg[m][n], X, NU), pv = sig * ds.pit[m][n];
        ss += g.glo[m] * g.glo[n] * sv * sv;
        pp += g.glo[m] * g.glo[n] * pv * pv;
      }
    diag_out[0] = tr.tau_pi * std::sqrt(std::max(ss, 0.0));
    diag_out[1] = std::sqrt(std::max(pp, 0.0)) / th.p;
    diag_out[2] = tr.tau_Pi * theta_out;
    diag_out[3] = std::fabs(Pi) / th.p;
  }
  return true;
}

/* ------------------------------------------------------------------------ freeze-out element (§5.10) ---- */
/* PAPER.md Eq. 145-148 (:1466-1482), per particle at the current state, given the rates k = dy/dx0 of Step 5:
     d_i eps   = (1/sigma*_a) sum_b m_b (eps_b - eps_a) d_i W_ab        ("derivatives ... using the SPH method", n = +1 form)
     d eps/dx0 = T ds/dx0 + mu_q dn_q/dx0 along the particle (first law), with s = S sigma, n_q = N_q sigma and
                 d sigma/dx0 = -sigma theta / gamma (D sigma = -sigma theta)
     d_0 eps   = d eps/dx0 - v^i d_i eps                                 (Eulerian time derivative)
     n_mu      = -d_mu eps / sqrt|d_mu eps d^mu eps|,   |d sigma| = m / (sigma |u^mu n_mu|)                       */
static void freezeout_element(const oracle_params& P, const Geometry& g, const State& y, const State& k, int64_t N,
                              Derived& d) {
  const int D = P.dim;
  for (int i = 0; i < 9; ++i) d.fo[i].assign(N, 0.0);
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t a = 0; a < N; ++a) {
    double de[4] = {0, 0, 0, 0};
    for (int64_t kk = d.nb_off[a]; kk < d.nb_off[a + 1]; ++kk) {
      const int64_t b = d.nb_idx[kk];
      double dr[3] = {0, 0, 0}, gW[3];
      for (int i = 0; i < D; ++i) dr[i] = y.f[OF_R1 + i][a] - y.f[OF_R1 + i][b];
      kernel_gradW(D, P.h, dr, gW);
      for (int i = 0; i < D; ++i) de[1 + i] += y.f[OF_MASS][b] * (d.th[b].e - d.th[a].e) * gW[i];
    }
    for (int i = 0; i < D; ++i) de[1 + i] /= d.sigma_star[a];
    double u[4];
    four_velocity(P, g, y, a, u);
    const double gam = u[0], sig = d.sigma[a], th_ = d.theta[a];
    const Thermo& th = d.th[a];
    const double dsig = -sig * th_ / gam;
    double deps = th.T * (sig * k.f[OF_S][a] + y.f[OF_S][a] * dsig);
    for (int q = 0; q < NQ; ++q) deps += th.mu[q] * (sig * k.f[OF_NB + q][a] + y.f[OF_NB + q][a] * dsig);
    de[0] = deps;
    for (int i = 1; i <= D; ++i) de[0] -= (u[i] / gam) * de[i];
    double nn = 0.0;
    for (int m = 0; m < 4; ++m) nn += g.gup[m] * de[m] * de[m];
    const double norm = std::sqrt(std::fabs(nn));
    double un = 0.0, nmu[4];
    for (int m = 0; m < 4; ++m) { nmu[m] = (norm > 0.0) ? -de[m] / norm : 0.0; un += u[m] * nmu[m]; }
    for (int m = 0; m < 4; ++m) { d.fo[m][a] = de[m]; d.fo[4 + m][a] = nmu[m]; }
    d.fo[8][a] = (un != 0.0) ? y.f[OF_MASS][a] / (sig * std::fabs(un)) : 0.0;
  }
}

/* f(y, x0): all of Steps 1-5 */
static double now_s() {
  return std::chrono::duration<double>(std::chrono::steady_clock::now().time_since_epoch()).count();
}

static int evaluate(oracle_ctx* c, const State& y, double x0, Derived& d, State& k) {
  const oracle_params& P = c->P;
  const int64_t N = c->N;
  const bool timing = std::getenv("ORACLE_TIMING") != nullptr;
  double t[6];
  t[0] = now_s();
  build_neighbours(P, y, N, d);
  t[1] = now_s();
  smoothing_sums(P, y, N, d);
  t[2] = now_s();
  thermo_pass(c, y, x0, d);
  t[3] = now_s();
  gradient_sums(P, y, N, d);
  t[4] = now_s();
  const Geometry g = geometry(P, x0);
  for (int f = 0; f < OF_NSTATE; ++f) k.f[f].assign(N, 0.0);
  d.theta.assign(N, 0.0);
  for (int i = 0; i < 4; ++i) d.diag[i].assign(N, 0.0);
  for (int i = 0; i < 3; ++i) d.fm[i].assign(N, 0.0);
  for (int q = 0; q < NQ; ++q) d.fk[q].assign(N, 0.0);
  int bad = 0;
#pragma omp parallel for schedule(dynamic, 16) reduction(+ : bad)
  for (int64_t a = 0; a < N; ++a) {
    double th = 0.0, dg[4] = {0.0, 0.0, 0.0, 0.0}, Isrc[7];
    for (int m = 0; m < 7; ++m) Isrc[m] = c->src[m].empty() ? 0.0 : c->src[m][a];
    if (P.dim == 2) Isrc[3] = 0.0;
    if (!eom_particle(P, g, y, d, a, x0, k, th, dg, Isrc)) bad++;
    d.theta[a] = th;
    for (int i = 0; i < 4; ++i) d.diag[i][a] = dg[i];
    for (int i = 0; i < P.dim; ++i) d.fm[i][a] = g.sqrtg * (d.FP[i][a] - d.FB[i][a]);
    for (int q = 0; q < NQ; ++q) d.fk[q][a] = -g.sqrtg * d.FK[q][a];
  }
  t[5] = now_s();
  if (timing)
    std::fprintf(stderr, "[oracle] N=%lld neighbours %.4f s, smoothing %.4f s, thermo %.4f s, gradient %.4f s, eom %.4f s\n",
                 (long long)N, t[1] - t[0], t[2] - t[1], t[3] - t[2], t[4] - t[3], t[5] - t[4]);
  if (bad) { c->err = "singular per-particle system"; return ORACLE_ERANGE; }
  return ORACLE_OK;
}

/* ---------------------------------------------------------------------------------------------- Step 6 ---- */
static void axpy(const State& y0, double a, const State& k, State& out, int64_t N) {
  for (int f = 0; f < OF_NSTATE; ++f) {
    out.f[f].resize(N);
    if (f == OF_MASS) { out.f[f] = y0.f[f]; continue; }
    for (int64_t i = 0; i < N; ++i) out.f[f][i] = y0.f[f][i] + a * k.f[f][i];
  }
}

static int rk_step(oracle_ctx* c) {
  const int64_t N = c->N;
  const double dt = c->P.dx0, x0 = c->x0;
  int rc;
  Derived& d = c->d;
  if (c->P.integrator == 2) {
    /* midpoint: k1 = f(y0, x0); y_half = y0 + dt/2 k1; k2 = f(y_half, x0 + dt/2); y1 = y0 + dt k2 */
    State k1, k2, yh;
    if ((rc = evaluate(c, c->y, x0, d, k1))) return rc;
    d.n_oob_steps += d.n_oob;
    axpy(c->y, 0.5 * dt, k1, yh, N);
    if ((rc = evaluate(c, yh, x0 + 0.5 * dt, d, k2))) return rc;
    d.n_oob_steps += d.n_oob;
    State y1;
    axpy(c->y, dt, k2, y1, N);
    c->y = y1;
  } else {
    /* classical RK4 */
    State k1, k2, k3, k4, t;
    if ((rc = evaluate(c, c->y, x0, d, k1))) return rc;
    d.n_oob_steps += d.n_oob;
    axpy(c->y, 0.5 * dt, k1, t, N);
    if ((rc = evaluate(c, t, x0 + 0.5 * dt, d, k2))) return rc;
    d.n_oob_steps += d.n_oob;
    axpy(c->y, 0.5 * dt, k2, t, N);
    if ((rc = evaluate(c, t, x0 + 0.5 * dt, d, k3))) return rc;
    d.n_oob_steps += d.n_oob;
    axpy(c->y, dt, k3, t, N);
    if ((rc = evaluate(c, t, x0 + dt, d, k4))) return rc;
    d.n_oob_steps += d.n_oob;
    State y1 = c->y;
    for (int f = 0; f < OF_NSTATE; ++f) {
      if (f == OF_MASS) continue;
      for (int64_t i = 0; i < N; ++i)
        y1.f[f][i] = c->y.f[f][i] + (dt / 6.0) * (k1.f[f][i] + 2.0 * k2.f[f][i] + 2.0 * k3.f[f][i] + k4.f[f][i]);
    }
    c->y = y1;
  }
  c->x0 = x0 + dt;
  c->derived_valid = false;
  return ORACLE_OK;
}

static int refresh(oracle_ctx* c) {
  if (c->derived_valid) return ORACLE_OK;
  int rc = evaluate(c, c->y, c->x0, c->d, c->rate);
  if (rc) return rc;
  freezeout_element(c->P, geometry(c->P, c->x0), c->y, c->rate, c->N, c->d);
  c->derived_valid = true;
  return ORACLE_OK;
}

}  // namespace

/* ================================================================================================ C ABI ==== */
extern "C" {

int oracle_create(const oracle_params* p, oracle_ctx** out) {
  if (!p || !out) return ORACLE_EINVAL;
  if ((p->dim != 2 && p->dim != 3) || (p->coords != 0 && p->coords != 1) || (p->integrator != 2 && p->integrator != 4) ||
      p->eom < 0 || p->eom > 2 || (p->eos_kind != 0 && p->eos_kind != 1) || !(p->h > 0.0) || !(p->dx0 > 0.0))
    return ORACLE_EINVAL;
  if (p->coords == 1 && !(p->x0_start > 0.0)) return ORACLE_EINVAL;
  oracle_ctx* c = new (std::nothrow) oracle_ctx();
  if (!c) return ORACLE_ENOMEM;
  c->P = *p;
  if (c->P.eom == 0) c->P.flags = 0;
  c->x0 = p->x0_start;
  *out = c;
  return ORACLE_OK;
}

int oracle_destroy(oracle_ctx* c) { delete c; return ORACLE_OK; }

const char* oracle_last_error(const oracle_ctx* c) { return c ? c->err.c_str() : "null context"; }

int oracle_load_particles(oracle_ctx* c, int64_t n, int32_t nfields, const int32_t* ids, const double* const* cols) {
  if (!c || n <= 0 || nfields <= 0 || !ids || !cols) return ORACLE_EINVAL;
  if (n > 2000000000LL) return ORACLE_EINVAL;
  for (int f = 0; f < OF_NSTATE; ++f) c->y.f[f].assign(n, (f == OF_MASS) ? 1.0 : 0.0);
  for (int k = 0; k < nfields; ++k) {
    const int id = ids[k];
    if (id < 0 || id >= OF_NSTATE || !cols[k]) { c->err = "bad field id in load"; return ORACLE_EINVAL; }
    std::copy(cols[k], cols[k] + n, c->y.f[id].begin());
  }
  /* fields of switched-off sectors are ignored (kept zero) */
  if (!shear_on(c->P)) for (int f = OF_PI11; f <= OF_PI33; ++f) c->y.f[f].assign(n, 0.0);
  if (!bulk_on(c->P)) c->y.f[OF_BULK].assign(n, 0.0);
  if (!diff_on(c->P)) for (int f = OF_JB1; f <= OF_JQ3; ++f) c->y.f[f].assign(n, 0.0);
  if (c->P.dim == 2) {
    c->y.f[OF_R3].assign(n, 0.0); c->y.f[OF_U3].assign(n, 0.0);
    c->y.f[OF_PI13].assign(n, 0.0); c->y.f[OF_PI23].assign(n, 0.0);
    c->y.f[OF_JB3].assign(n, 0.0); c->y.f[OF_JS3].assign(n, 0.0); c->y.f[OF_JQ3].assign(n, 0.0);
  }
  c->N = n;
  for (int m = 0; m < 7; ++m) c->src[m].clear();
  c->d.n_oob_steps = 0;
  c->x0 = c->P.x0_start;
  c->loaded = true;
  c->derived_valid = false;
  return ORACLE_OK;
}

int oracle_load_eos_table(oracle_ctx* c, const int32_t dims[4], const int32_t axis_kind[4], const double* const axes[4],
                          int32_t ncols, const int32_t* col_ids, const double* data) {
  if (!c || !dims || !axis_kind || !axes || !col_ids || !data || ncols <= 0 || ncols > NCOLMAX) return ORACLE_EINVAL;
  Table& tb = c->tab;
  int64_t nodes = 1;
  for (int k = 0; k < 4; ++k) {
    if (dims[k] < 2 || !axes[k] || (axis_kind[k] != 0 && axis_kind[k] != 1)) return ORACLE_EINVAL;
    if (k == 0 && axis_kind[k] != 0) return ORACLE_EINVAL;
    tb.dims[k] = dims[k]; tb.kind[k] = axis_kind[k];
    tb.ax[k].assign(axes[k], axes[k] + dims[k]);
    for (int i = 1; i < dims[k]; ++i) if (!(tb.ax[k][i] > tb.ax[k][i - 1])) { c->err = "axis not increasing"; return ORACLE_EINVAL; }
    nodes *= dims[k];
  }
  for (int cc = 0; cc < NCOLMAX; ++cc) tb.col_of[cc] = -1;
  for (int k = 0; k < ncols; ++k) {
    if (col_ids[k] < 0 || col_ids[k] >= NCOLMAX) return ORACLE_EINVAL;
    tb.col_of[col_ids[k]] = k;
  }
  for (int cc = 0; cc <= C_WS; ++cc) if (tb.col_of[cc] < 0) { c->err = "table lacks a required column"; return ORACLE_EINVAL; }
  if (diff_on(c->P)) for (int cc = C_WB; cc <= C_WQ; ++cc) if (tb.col_of[cc] < 0) { c->err = "diffusion needs dw/dn_q columns"; return ORACLE_EINVAL; }
  tb.ncols = ncols;
  tb.data.assign(data, data + nodes * ncols);
  tb.loaded = true;
  c->derived_valid = false;
  return ORACLE_OK;
}

int oracle_step(oracle_ctx* c, int32_t nsteps) {
  if (!c || nsteps < 0) return ORACLE_EINVAL;
  if (!c->loaded || (c->P.eos_kind == 1 && !c->tab.loaded)) { if (c) c->err = "step before load"; return ORACLE_ESTATE; }
  for (int s = 0; s < nsteps; ++s) {
    int rc = rk_step(c);
    if (rc) return rc;
  }
  return ORACLE_OK;
}

int oracle_read_fields(oracle_ctx* c, int32_t nfields, const int32_t* ids, double* const* cols, int64_t capacity) {
  if (!c || nfields <= 0 || !ids || !cols) return ORACLE_EINVAL;
  if (!c->loaded) return ORACLE_ESTATE;
  if (capacity < c->N) return ORACLE_EINVAL;
  bool need_derived = false;
  for (int k = 0; k < nfields; ++k) if (ids[k] >= OF_NSTATE) need_derived = true;
  if (need_derived) {
    if (c->P.eos_kind == 1 && !c->tab.loaded) return ORACLE_ESTATE;
    int rc = refresh(c);
    if (rc) return rc;
  }
  const Derived& d = c->d;
  for (int k = 0; k < nfields; ++k) {
    const int id = ids[k];
    const std::vector<double>* src = nullptr;
    std::vector<double> tmp;
    if (id >= 0 && id < OF_NSTATE) src = &c->y.f[id];
    else if (id >= OF_RATE && id < OF_RATE + OF_NSTATE) src = &c->rate.f[id - OF_RATE];
    else switch (id) {
      case OF_SIGMA_STAR: src = &d.sigma_star; break;
      case OF_S_DENS: src = &d.s; break;
      case OF_RHO_B: src = &d.n[0]; break;
      case OF_RHO_S: src = &d.n[1]; break;
      case OF_RHO_Q: src = &d.n[2]; break;
      case OF_GAMMA: src = &d.gamma; break;
      case OF_NNB: src = &d.nnb; break;
      case OF_CELL: src = &d.cell; break;
      case OF_THETA: src = &d.theta; break;
      case OF_FO_DE0: case OF_FO_DE1: case OF_FO_DE2: case OF_FO_DE3: case OF_FO_N0: case OF_FO_N1: case OF_FO_N2:
      case OF_FO_N3: case OF_FO_DSIGMA: src = &d.fo[id - OF_FO_DE0]; break;
      case OF_KN_PI: src = &d.diag[0]; break;
      case OF_RE_PI: src = &d.diag[1]; break;
      case OF_KN_BULK: src = &d.diag[2]; break;
      case OF_RE_BULK: src = &d.diag[3]; break;
      case OF_SIGMA: src = &d.sigma; break;
      case OF_S_STAR: src = &d.s_star; break;
      case OF_RHOSTAR_B: src = &d.rho_star[0]; break;
      case OF_RHOSTAR_S: src = &d.rho_star[1]; break;
      case OF_RHOSTAR_Q: src = &d.rho_star[2]; break;
      case OF_DIVV: src = &d.divv; break;
      case OF_FM1: src = &d.fm[0]; break;
      case OF_FM2: src = &d.fm[1]; break;
      case OF_FM3: src = &d.fm[2]; break;
      case OF_FK_B: src = &d.fk[0]; break;
      case OF_FK_S: src = &d.fk[1]; break;
      case OF_FK_Q: src = &d.fk[2]; break;
      case OF_T: case OF_MU_B: case OF_MU_S: case OF_MU_Q: case OF_P: case OF_E: case OF_CS2: case OF_WS:
        tmp.resize(c->N);
        for (int64_t a = 0; a < c->N; ++a) {
          const Thermo& th = d.th[a];
          tmp[a] = (id == OF_T) ? th.T : (id == OF_MU_B) ? th.mu[0] : (id == OF_MU_S) ? th.mu[1] : (id == OF_MU_Q) ? th.mu[2]
                 : (id == OF_P) ? th.p : (id == OF_E) ? th.e : (id == OF_CS2) ? th.cs2 : th.ws;
        }
        src = &tmp;
        break;
      default: c->err = "bad field id in read"; return ORACLE_EINVAL;
    }
    if (!cols[k]) return ORACLE_EINVAL;
    std::copy(src->begin(), src->begin() + c->N, cols[k]);
  }
  return ORACLE_OK;
}

/* Step 7 */
int oracle_conserved_totals(oracle_ctx* c, double out[16]) {
  if (!c || !out) return ORACLE_EINVAL;
  if (!c->loaded) return ORACLE_ESTATE;
  int rc = refresh(c);
  if (rc) return rc;
  const oracle_params& P = c->P;
  const Geometry g = geometry(P, c->x0);
  const Derived& d = c->d;
  for (int k = 0; k < 16; ++k) out[k] = 0.0;
  double E = 0, Pm[3] = {0, 0, 0}, St = 0, Nq[NQ] = {0, 0, 0}, M = 0, work = 0, trace = 0, npairs = 0;
  for (int64_t a = 0; a < c->N; ++a) {
    double u[4];
    four_velocity(P, g, c->y, a, u);
    const double gam = u[0], sig = d.sigma[a], m = c->y.f[OF_MASS][a];
    const Thermo& th = d.th[a];
    const Dissip ds = dissipative(P, g, c->y, a, u);
    const double w = th.e + th.p, Pi = ds.bulkt * sig;
    const double Cc = (w + Pi) / sig;
    St += m * c->y.f[OF_S][a];
    for (int q = 0; q < NQ; ++q) Nq[q] += m * (c->y.f[OF_NB + q][a] + ds.Jt[q][0] / gam);
    for (int i = 1; i <= P.dim; ++i) Pm[i - 1] += m * (Cc * g.glo[i] * u[i] + g.glo[i] * ds.pit[0][i] / gam);
    /* T^{00} = (w + Pi) gamma^2 - (p + Pi) g^{00} + pi^{00} */
    const double T00 = (w + Pi) * gam * gam - (th.p + Pi) + sig * ds.pit[0][0];
    const double vol = m / d.sigma_star[a];
    if (P.coords == 1 && P.dim == 3) {
      const double eta = c->y.f[OF_R3][a];
      const double T03 = (w + Pi) * gam * u[3] + sig * ds.pit[0][3];
      E += vol * g.sqrtg * (T00 * std::cosh(eta) + c->x0 * T03 * std::sinh(eta));
    } else {
      E += vol * g.sqrtg * T00;
    }
    M += m;
    work += c->y.f[OF_WORK][a];
    double tr = ds.pit[0][0];
    for (int i = 1; i <= 3; ++i) tr += g.glo[i] * ds.pit[i][i];
    trace = std::max(trace, std::fabs(tr * sig));
    npairs += d.nnb[a];
  }
  out[0] = c->x0; out[1] = E; out[2] = Pm[0]; out[3] = Pm[1]; out[4] = Pm[2]; out[5] = St;
  out[6] = Nq[0]; out[7] = Nq[1]; out[8] = Nq[2]; out[9] = M; out[10] = work; out[11] = (double)d.n_oob;
  out[12] = trace; out[13] = 0.0; out[14] = npairs; out[15] = (double)d.n_oob_steps;
  return ORACLE_OK;
}

int oracle_read_neighbors(oracle_ctx* c, int64_t* counts, int64_t* offsets, int32_t* list, int64_t cap) {
  if (!c || !counts) return ORACLE_EINVAL;
  if (!c->loaded) return ORACLE_ESTATE;
  int rc = refresh(c);
  if (rc) return rc;
  const Derived& d = c->d;
  for (int64_t a = 0; a < c->N; ++a) counts[a] = d.nb_off[a + 1] - d.nb_off[a];
  if (offsets) for (int64_t a = 0; a <= c->N; ++a) offsets[a] = d.nb_off[a];
  if (list) {
    if (cap < d.nb_off[c->N]) return ORACLE_EINVAL;
    std::copy(d.nb_idx.begin(), d.nb_idx.end(), list);
  }
  return ORACLE_OK;
}

double oracle_kernel_W(int32_t D, double h, double r) { return kernel_W(D, h, r); }
void oracle_kernel_gradW(int32_t D, double h, const double dr[3], double out[3]) { kernel_gradW(D, h, dr, out); }

static void thermo_to_out(const Thermo& th, double out[11]) {
  out[C_T] = th.T; out[C_MUB] = th.mu[0]; out[C_MUS] = th.mu[1]; out[C_MUQ] = th.mu[2]; out[C_P] = th.p;
  out[C_CS2] = th.cs2; out[C_E] = th.e; out[C_WS] = th.ws; out[C_WB] = th.wq[0]; out[C_WSQ] = th.wq[1]; out[C_WQ] = th.wq[2];
}

int oracle_eos_closed_form(const oracle_params* p, double s, const double n[3], double out[11]) {
  if (!p || !n || !out) return ORACLE_EINVAL;
  thermo_to_out(eos_closed_form(*p, s, n), out);
  return ORACLE_OK;
}

int oracle_eos_forward(const oracle_params* p, double T, const double mu[3], double out[5]) {
  if (!p || !mu || !out) return ORACLE_EINVAL;
  double pp, s, n[NQ];
  eos_forward(*p, T, mu, pp, s, n);
  out[0] = pp; out[1] = s; out[2] = n[0]; out[3] = n[1]; out[4] = n[2];
  return ORACLE_OK;
}

int oracle_eos_table_lookup(oracle_ctx* c, double s, const double n[3], double out[11], int32_t* oob) {
  if (!c || !n || !out) return ORACLE_EINVAL;
  if (!c->tab.loaded) return ORACLE_ESTATE;
  const Thermo th = eos_table(c->tab, s, n);
  thermo_to_out(th, out);
  if (oob) *oob = th.oob;
  return ORACLE_OK;
}

int oracle_invert_forward_table(const oracle_params* p, const int32_t fdims[4], const double* const faxes[4], const double* fdata,
                                int64_t nt, const double* s, const double* const n[3], double* out, int32_t* flag, int32_t* iters) {
  if (!p || !fdims || !faxes || !fdata || nt < 0 || !s || !n || !out || !flag) return ORACLE_EINVAL;
  FwdTable ft;
  for (int k = 0; k < 4; ++k) {
    if (fdims[k] < 2 || !faxes[k]) return ORACLE_EINVAL;
    for (int i = 1; i < fdims[k]; ++i) if (!(faxes[k][i] > faxes[k][i - 1])) return ORACLE_EINVAL;
    ft.dims[k] = fdims[k];
    ft.ax[k] = faxes[k];
  }
  ft.data = fdata;
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t a = 0; a < nt; ++a) {
    const double nn[NQ] = {n[0][a], n[1][a], n[2][a]};
    int32_t f = 0, it = 0;
    const Thermo th = invert_forward_point(*p, ft, s[a], nn, f, it);
    thermo_to_out(th, out + a * 11);
    flag[a] = f;
    if (iters) iters[a] = it;
  }
  return ORACLE_OK;
}

int oracle_set_sources(oracle_ctx* c, const double* const I[4], const double* const Iq[3]) {
  if (!c) return ORACLE_EINVAL;
  if (!c->loaded) return ORACLE_ESTATE;
  for (int m = 0; m < 7; ++m) {
    const double* col = (m < 4) ? (I ? I[m] : nullptr) : (Iq ? Iq[m - 4] : nullptr);
    if (col) c->src[m].assign(col, col + c->N);
    else c->src[m].clear();
  }
  c->derived_valid = false;
  return ORACLE_OK;
}

int oracle_smear_sources(oracle_ctx* c, int64_t np, const double* const p[4], const double* const r[3], const double* t,
                         double h_source, double eta_norm, double* const j[4]) {
  if (!c || np < 0 || !p || !r || !t || !j || !(h_source > 0.0)) return ORACLE_EINVAL;
  if (!c->loaded) return ORACLE_ESTATE;
  const int D = c->P.dim;
  const Geometry g = geometry(c->P, c->x0);
  const double x0 = c->x0, dx0 = c->P.dx0;
  const double pref = eta_norm / (dx0 * g.sqrtg);
  for (int64_t i = 0; i < c->N; ++i) {
    double acc[4] = {0, 0, 0, 0};
    for (int64_t k = 0; k < np; ++k) {
      if (!(t[k] > x0 - dx0 && t[k] <= x0)) continue;            /* Eq. 35: x0 - dx0 < t_k <= x0 */
      double r2 = 0.0;
      for (int a = 0; a < D; ++a) { const double dr = c->y.f[OF_R1 + a][i] - r[a][k]; r2 += dr * dr; }
      const double W = kernel_W(D, h_source, std::sqrt(r2));
      for (int m = 0; m < 4; ++m) acc[m] += p[m][k] * W;
    }
    for (int m = 0; m < 4; ++m) j[m][i] = pref * acc[m];
  }
  return ORACLE_OK;
}

}  /* extern "C" */
