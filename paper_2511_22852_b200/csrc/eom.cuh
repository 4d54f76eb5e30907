/*
 * csrc/eom.cuh — steps a7 (equations of motion) and a8 (RK stage update).
 *
 * PAPER.md Eq. 87-95 (:964-988): the time derivatives of phi_a enter linearly, M dphi/dx0 = F, and the system
 * reduces to a D x D solve for du^i/dx0 (Eq. 95).  The reduction used here: GIVEN a trial du^i/dx0, every other
 * rate is explicit —
 *     du^0                      from u.u = 1 (Eq. 97 :1011)
 *     theta, Du^mu, sigma^{mu nu}, omega^{mu nu}   from du^mu and the SPH gradients (Notation :164-169)
 *     d(Pi/sigma)               bulk relaxation, Eq. 49 :676 / Eq. 52 row 1
 *     d(pi^{ij}/sigma)          shear relaxation, Eq. 50 :678 / Eq. 52 row 3
 *     d(J^i_q/sigma)            diffusion relaxation, Eq. 51 :680
 *     d(pi^{0 mu}/sigma), d(J^0_q/sigma)   from the orthogonality constraints
 *     dN_q                      charge conservation,  dS  entropy production (Eq. 96 :1003, Eq. 98 :1016)
 * — so the momentum equation  d/dx0[ C u_i + pi~^0_i / gamma ] = sqrt(-g)(FP_i - FB_i)  is an affine map
 * residual(du) = r0 + M du.  The kernel evaluates the residual at du = 0 and at the D unit vectors (columns of M,
 * = the matrix of Eq. 95), solves M du = -r0 by Gaussian elimination with partial pivoting on the D x D matrix,
 * and evaluates the explicit rates once more at the solution.  No dense system in all 17/23 unknowns is formed.
 *
 * The metric is diagonal, g = diag(1,-1,-1,-G3); the only Christoffel symbols are Gamma^tau_{eta eta} = tau,
 * Gamma^eta_{tau eta} = 1/tau (:488), which are written out explicitly.
 */
#pragma once
#include "common.cuh"
#include "thermo_eos.cuh"

namespace ccake {

struct EomIn {
  double u[4], ulo[4], v[4], glo[4], gup[4];
  double gam, sig, sst, T, mu[NQ], p, e, cs2, ws, wq[NQ], s;
  /* reciprocals, taken once per particle (a double division is ~25 instructions; the rate evaluation runs D + 2
     times): 1/gamma, 1/tau, 1/sigma, 1/(tau_Pi sigma gamma), 1/(sigma tau_pi), 1/(tau_q sigma), 1/(gamma sigma T) */
  double igam, itau, isig, i_tauPi_sig_gam, i_sig_taupi, i_tauq_sig[NQ], i_gam_sig_T;
  double eta, zeta, tau_pi, tau_Pi, kappa[NQ][NQ], tau_q[NQ];
  double delta_PiPi, lambda_Pipi, delta_pipi, tau_pipi, lambda_piPi, phi_omega;
  double CDc[4][4];      /* nabla_mu u^nu without the du^nu part of the row mu = 0 */
  double Duc[4];         /* u^mu CDc[mu][nu] */
  double thc;            /* gamma (div v + Gamma_g) */
  double rhsJ[NQ][3];    /* constant right-hand side of the diffusion equation */
  double FM[3];          /* sqrt(-g) (FP_i - FB_i) */
  double FKs[NQ];        /* sqrt(-g) FK_q - I_q / (gamma sigma) */
  double uI;             /* u_mu I^mu, source of the entropy equation (Eq. 96); 0 without sources */
  Dissip ds;
};

struct EomOut {
  double du0, theta, dS, dN[NQ], dBulk, dpit[4][4], dJt[NQ][4], res[3];
};

/* MODE 0: the rates at a given du.  MODE 1: at du = 0 (a literal, so every du term folds away).  MODE 2 + c: the
   HOMOGENEOUS part of the affine map at the unit vector e_c — every term without du is dropped (K = 0 below) and the
   zeros of e_c fold away, so res is column c of the matrix of Eq. 95 directly (no difference of two evaluations). */
template <int D, int MODE>
__device__ __forceinline__ void eom_rates(const KParams& kp, const Geom& gm, const EomIn& in, const double du_in[3],
                                          EomOut& o, double* sgsq_out = nullptr) {
  constexpr bool H = MODE >= 2;
  constexpr double K = H ? 0.0 : 1.0;            /* multiplies the du-independent terms */
  const double gam = in.gam, sig = in.sig;
  const double igam = in.igam, itau = in.itau;
  double du[4], dulo[4];
  if (MODE == 0) { du[1] = du_in[0]; du[2] = du_in[1]; du[3] = (D == 3) ? du_in[2] : 0.0; }
  else { du[1] = (MODE == 2) ? 1.0 : 0.0; du[2] = (MODE == 3) ? 1.0 : 0.0; du[3] = (MODE == 4) ? 1.0 : 0.0; }
  /* Eq. 97, nu = 0: u_0 du^0 = -u_k du^k - (1/2) u^a u^b dg_ab/dx0,  dg_33/dx0 = -dG3 */
  const double gt = H ? 0.0 : -in.u[3] * in.u[3] * gm.dG3;
  du[0] = -(in.ulo[1] * du[1] + in.ulo[2] * du[2] + in.ulo[3] * du[3]) * igam - gt * (0.5 * igam);
#pragma unroll
  for (int m = 0; m < 4; ++m) dulo[m] = in.glo[m] * du[m];
  if (!H) dulo[3] += -gm.dG3 * in.u[3];
  o.du0 = du[0];
  const double theta = H ? du[0] : in.thc + du[0];
  o.theta = theta;
  /* covariant derivative, acceleration */
  double CD[4][4], Du[4], Dulo[4];
#pragma unroll
  for (int m = 0; m < 4; ++m)
#pragma unroll
    for (int n = 0; n < 4; ++n) CD[m][n] = H ? 0.0 : in.CDc[m][n];
#pragma unroll
  for (int n = 0; n < 4; ++n) { CD[0][n] += du[n]; Du[n] = (H ? 0.0 : in.Duc[n]) + gam * du[n]; Dulo[n] = in.glo[n] * Du[n]; }

  const double Pi = in.ds.bulkt * sig;
  const bool need_sg = kp.shear || (kp.bulk && in.lambda_Pipi != 0.0) || sgsq_out != nullptr;
  double sg[4][4];
  if (need_sg) {
#pragma unroll
    for (int m = 0; m < 4; ++m)
#pragma unroll
      for (int n = m; n < 4; ++n) {
        const double Delta = ((m == n) ? in.gup[m] : 0.0) - in.u[m] * in.u[n];
        const double v = 0.5 * (in.gup[m] * CD[m][n] + in.gup[n] * CD[n][m]) - 0.5 * (in.u[m] * Du[n] + in.u[n] * Du[m]) -
                         (Delta * (1.0 / 3.0)) * theta;
        sg[m][n] = v; sg[n][m] = v;
      }
  }
  if (sgsq_out) {                                  /* sigma^{mn} sigma_{mn} for Eq. 58 (diagonal metric) */
    double ss = 0.0;
#pragma unroll
    for (int m = 0; m < 4; ++m)
#pragma unroll
      for (int n = 0; n < 4; ++n) ss += in.glo[m] * in.glo[n] * sg[m][n] * sg[m][n];
    *sgsq_out = ss;
  }
  /* bulk */
  o.dBulk = 0.0;
  if (kp.bulk) {
    double rhs = -K * Pi - in.zeta * theta + (in.tau_Pi - in.delta_PiPi) * Pi * theta;
    if (in.lambda_Pipi != 0.0) {
      double acc = 0.0;
#pragma unroll
      for (int m = 0; m < 4; ++m)
#pragma unroll
        for (int n = 0; n < 4; ++n) acc += sig * in.ds.pit[m][n] * in.glo[m] * in.glo[n] * sg[m][n];
      rhs += in.lambda_Pipi * acc;
    }
    o.dBulk = rhs * in.i_tauPi_sig_gam;
  }
  /* shear */
#pragma unroll
  for (int m = 0; m < 4; ++m)
#pragma unroll
    for (int n = 0; n < 4; ++n) o.dpit[m][n] = 0.0;
  if (kp.shear) {
    double om[4][4];
    const bool need_om = in.phi_omega != 0.0;
    if (need_om)
#pragma unroll
      for (int m = 0; m < 4; ++m)
#pragma unroll
        for (int n = 0; n < 4; ++n)
          om[m][n] = 0.5 * (in.gup[m] * CD[m][n] - in.gup[n] * CD[n][m]) - 0.5 * (in.u[m] * Du[n] - in.u[n] * Du[m]);
    double Xtr = 0.0;
    if (in.tau_pipi != 0.0)
#pragma unroll
      for (int l = 0; l < 4; ++l)
#pragma unroll
        for (int m = 0; m < 4; ++m) Xtr += sig * in.ds.pit[l][m] * in.glo[l] * in.glo[m] * sg[m][l];
#pragma unroll
    for (int i = 1; i <= 3; ++i)
#pragma unroll
      for (int j = i; j <= 3; ++j) {
        if (D == 2 && j == 3 && i != 3) continue;          /* pi^{13}, pi^{23} vanish by symmetry in 2+1D */
        double conn = 0.0;                                  /* u^l Gamma^i_{l r} pi~^{r j} + (i <-> j)      */
        if (gm.hyper && !H) {
          if (i == 3) conn += (gam * in.ds.pit[3][j] + in.u[3] * in.ds.pit[0][j]) * itau;
          if (j == 3) conn += (gam * in.ds.pit[i][3] + in.u[3] * in.ds.pit[i][0]) * itau;
        }
        double acc = 0.0;
#pragma unroll
        for (int l = 0; l < 4; ++l) acc += (in.u[i] * in.ds.pit[j][l] + in.u[j] * in.ds.pit[i][l]) * Dulo[l];
        const double piij = sig * in.ds.pit[i][j];
        double rhs = -K * piij + 2.0 * in.eta * sg[i][j] + (in.tau_pi - in.delta_pipi) * piij * theta;
        if (in.tau_pipi != 0.0) {
          double X = 0.0;
#pragma unroll
          for (int l = 0; l < 4; ++l) {
            X += 0.5 * sig * in.ds.pit[l][i] * in.glo[l] * sg[l][j];
            X += 0.5 * sig * in.ds.pit[l][j] * in.glo[l] * sg[l][i];
          }
          const double Delta = ((i == j) ? in.gup[i] : 0.0) - in.u[i] * in.u[j];
          X -= (Delta * (1.0 / 3.0)) * Xtr;
          rhs -= in.tau_pipi * X;
        }
        if (in.lambda_piPi != 0.0) rhs += in.lambda_piPi * Pi * sg[i][j];
        if (need_om) {
          double Yv = 0.0;
#pragma unroll
          for (int l = 0; l < 4; ++l) {
            Yv += 0.5 * sig * in.ds.pit[i][l] * in.glo[l] * om[j][l];
            Yv += 0.5 * sig * in.ds.pit[j][l] * in.glo[l] * om[i][l];
          }
          rhs += 2.0 * in.tau_pi * in.phi_omega * Yv;
        }
        const double d = (rhs * in.i_sig_taupi - conn - acc) * igam;
        o.dpit[i][j] = d; o.dpit[j][i] = d;
      }
    /* d/dx0 of u_mu pi~^{mu nu} = 0 */
#pragma unroll
    for (int n = 1; n <= 3; ++n) {
      double acc = 0.0;
#pragma unroll
      for (int m = 0; m < 4; ++m) acc -= dulo[m] * in.ds.pit[m][n];
#pragma unroll
      for (int j = 1; j <= 3; ++j) acc -= in.ulo[j] * o.dpit[j][n];
      o.dpit[0][n] = acc * igam; o.dpit[n][0] = acc * igam;
    }
    double acc = 0.0;
#pragma unroll
    for (int m = 0; m < 4; ++m) acc -= dulo[m] * in.ds.pit[m][0];
#pragma unroll
    for (int j = 1; j <= 3; ++j) acc -= in.ulo[j] * o.dpit[j][0];
    o.dpit[0][0] = acc * igam;
  }
  /* diffusion */
#pragma unroll
  for (int q = 0; q < NQ; ++q)
#pragma unroll
    for (int m = 0; m < 4; ++m) o.dJt[q][m] = 0.0;
  if (kp.diff) {
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
      double JDu = 0.0;
#pragma unroll
      for (int n = 0; n < 4; ++n) JDu += in.ds.Jt[q][n] * Dulo[n];
#pragma unroll
      for (int i = 1; i <= D; ++i) {
        double conn = 0.0;
        if (gm.hyper && i == 3 && !H) conn = (gam * in.ds.Jt[q][3] + in.u[3] * in.ds.Jt[q][0]) * itau;
        o.dJt[q][i] = (H ? -in.u[i] * JDu : in.rhsJ[q][i - 1] * in.i_tauq_sig[q] - conn - in.u[i] * JDu) * igam;
      }
      double acc = 0.0;
#pragma unroll
      for (int m = 0; m < 4; ++m) acc -= dulo[m] * in.ds.Jt[q][m];
#pragma unroll
      for (int j = 1; j <= 3; ++j) acc -= in.ulo[j] * o.dJt[q][j];
      o.dJt[q][0] = acc * igam;
    }
  }
  /* charge: d/dx0 [ N_q + J~^0_q / gamma ] = -sqrt(-g) FK_q */
#pragma unroll
  for (int q = 0; q < NQ; ++q)
    o.dN[q] = -K * in.FKs[q] - o.dJt[q][0] * igam + (in.ds.Jt[q][0] * (igam * igam)) * du[0];
  /* entropy, Eq. 96: gamma sigma (T dS + mu_q dN_q) = -Pi theta + pi^mu_nu nabla_mu u^nu */
  {
    double rhs = -Pi * theta + K * in.uI;
    if (kp.shear)
#pragma unroll
      for (int m = 0; m < 4; ++m)
#pragma unroll
        for (int n = 0; n < 4; ++n) rhs += sig * in.ds.pit[m][n] * in.glo[n] * CD[m][n];
    double lhs = 0.0;
#pragma unroll
    for (int q = 0; q < NQ; ++q) lhs += gam * sig * in.mu[q] * o.dN[q];
    o.dS = (rhs - lhs) * in.i_gam_sig_T;
  }
  /* momentum residual */
  const double w = in.e + in.p;
  const double A = w * in.cs2;
  const double Cc = w * in.isig + in.ds.bulkt;
  double dC = in.ws * o.dS + o.dBulk - (A * in.isig) * (theta * igam);
#pragma unroll
  for (int q = 0; q < NQ; ++q) dC += in.wq[q] * o.dN[q];
#pragma unroll
  for (int i = 1; i <= D; ++i) {
    const double pit0_lo = in.glo[i] * in.ds.pit[0][i];
    double dpit0_lo = in.glo[i] * o.dpit[0][i];
    if (i == 3 && !H) dpit0_lo += -gm.dG3 * in.ds.pit[0][3];
    o.res[i - 1] = in.ulo[i] * dC + Cc * dulo[i] + dpit0_lo * igam - (pit0_lo * (igam * igam)) * du[0] - K * in.FM[i - 1];
  }
}

/* RK bookkeeping of one substep (DESIGN reading 7):
     y_out = y_base + c_out * k                 (stage state, or the final state for RK2)
     RK4:  acc = k (mode 1) | acc + w k (mode 2) ; final: y_out = y_base + c_out * (acc + w k) (mode 3)          */
struct RkArgs {
  const double* Ycur;   /* state the rates are evaluated at        */
  const double* Ybase;  /* y0 of the step                          */
  double* Yout;         /* may alias Ybase (own-slot read then write) */
  double* Yacc;         /* RK4 accumulator or NULL                 */
  double* Krate;        /* rates in store order, or NULL           */
  double* theta_out;    /* sorted order                            */
  double* diag;         /* 4 x npad, sorted order: Kn_pi, Re_pi^-1, Kn_Pi, Re_Pi^-1 (DIAG kernels only) */
  const double* src;    /* 7 x npad, ORIGINAL particle order: I^0..I^3, I_B, I_S, I_Q (ccake_set_sources), or NULL */
  const uint32_t* orig; /* store slot -> original (load) index: for src, and to tell ghosts */
  int64_t n_own;        /* load indices >= n_own are ghost particles of a slab context (slab.cuh): evolved like the rest, but
                           their rates are not valid and not checked (their state is re-imported before every substep) */
  double c_out, w_acc;
  int acc_mode;         /* 0 none | 1 set | 2 add | 3 final        */
  int update;           /* 0: rates only (refresh)                 */
};

/* CCAKE_EOM_COMBINE (default): the rates at the solution are out(0) + sum_c du_c * (homogeneous part at e_c), from the stored
   outputs of the evaluations that built the D x D system, instead of one more general evaluation: 1.35 -> 1.28 ms per substep on
   C4.  (The DIAG instantiation keeps the general evaluation: it needs sigma^{mn} at the solution.) */
#ifndef CCAKE_EOM_NO_COMBINE
#define CCAKE_EOM_COMBINE 1
#endif
/* resident blocks per SM the register budget is set for.  3-D (C4): 2 -> 1.57 ms, 3 -> 1.41, 4 -> 1.35, 5 -> 1.64, 6 -> 1.98 per
   substep; 2-D (C3): 2 -> 0.130 ms, 3 -> 0.111, 4 -> 0.105 */
#ifndef CCAKE_EOM_MINB3
#define CCAKE_EOM_MINB3 4
#endif
#ifndef CCAKE_EOM_MINB2
#define CCAKE_EOM_MINB2 4
#endif
template <int D, bool DIAG>
__global__ void __launch_bounds__(128, (D == 3) ? CCAKE_EOM_MINB3 : CCAKE_EOM_MINB2)
eom_kernel(int64_t n, KParams kp, const double* __restrict__ x0_dev, double x0_off, int64_t npad, Sorted so, RkArgs rk,
           uint32_t field_mask, Status* __restrict__ status) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= n) return;
  const Geom gm = make_geom(kp.coords, *x0_dev + x0_off);      /* as the thermo kernel: time of this substep from device memory */
  const int64_t a = so.perm[i];
  const double* Y = rk.Ycur;          /* may alias rk.Yout (RK4 stages 2, 3: own slot read, then written): no __restrict__ */
  EomIn in;
  load_u(kp, gm, Y, npad, a, in.u);
  in.gam = in.u[0];
  in.igam = 1.0 / in.gam;
  in.itau = gm.hyper ? 1.0 / gm.tau : 0.0;
  in.glo[0] = 1.0; in.glo[1] = -1.0; in.glo[2] = -1.0; in.glo[3] = -gm.G3;
#pragma unroll
  for (int m = 0; m < 4; ++m) { in.gup[m] = (m == 3) ? -1.0 / gm.G3 : in.glo[m]; in.ulo[m] = in.glo[m] * in.u[m]; in.v[m] = in.u[m] * in.igam; }
  load_dissip<D>(kp, gm, Y, npad, a, in.u, in.ds);
  in.sig = so.sigma[i]; in.sst = so.sigma_star[i]; in.s = so.s[i];
  in.T = so.T[i]; in.p = so.p[i]; in.e = so.e[i]; in.cs2 = so.cs2[i]; in.ws = so.ws[i];
#pragma unroll
  for (int q = 0; q < NQ; ++q) { in.mu[q] = so.mu[q][i]; in.wq[q] = so.wq[q][i]; }
  /* transport coefficients, §5.3 (:732-769), DESIGN reading 11 */
  {
    const double w = in.e + in.p;
    in.eta = kp.eta_over_s * in.s;
    in.tau_pi = fmax(kp.tau_pi_coeff * in.eta / w, kp.tau_floor);
    const double dT = in.T - kp.zeta_T_peak;
    in.zeta = (kp.zeta_width > 0.0)
                  ? kp.zeta_max * (kp.zeta_width * kp.zeta_width) / (kp.zeta_width * kp.zeta_width + dT * dT) * in.s
                  : kp.zeta_max * in.s;
    in.tau_Pi = kp.tau_Pi_coeff * in.tau_pi;
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
#pragma unroll
      for (int r = 0; r < NQ; ++r) in.kappa[q][r] = kp.kappa_over_T2[q * 3 + r] * in.T * in.T;
      in.tau_q[q] = kp.tau_q_times_T[q] / in.T;
    }
    in.delta_PiPi = in.tau_Pi; in.lambda_Pipi = 0.0; in.delta_pipi = (4.0 / 3.0) * in.tau_pi; in.tau_pipi = 0.0;
    in.lambda_piPi = 0.0; in.phi_omega = 0.0;
    if (kp.eom == 2) {
      in.delta_PiPi = kp.dnmr[0] * in.tau_Pi; in.lambda_Pipi = kp.dnmr[1] * in.tau_Pi;
      in.delta_pipi = kp.dnmr[2] * in.tau_pi; in.tau_pipi = kp.dnmr[3] * in.tau_pi;
      in.lambda_piPi = kp.dnmr[4]; in.phi_omega = kp.dnmr[5];
    }
  in.isig = 1.0 / in.sig;
  in.i_tauPi_sig_gam = 1.0 / (in.tau_Pi * in.sig * in.gam);
  in.i_sig_taupi = 1.0 / (in.sig * in.tau_pi);
#pragma unroll
  for (int q = 0; q < NQ; ++q) in.i_tauq_sig[q] = 1.0 / (in.tau_q[q] * in.sig);
  in.i_gam_sig_T = 1.0 / (in.gam * in.sig * in.T);
  }
  /* gradients: d_k u^j from the SPH sums, d_k u^0 from u_mu d_k u^mu = 0, d_0 = d/dx0 - v^k d_k */
  {
    double PU[4][4];
#pragma unroll
    for (int m = 0; m < 4; ++m)
#pragma unroll
      for (int nn = 0; nn < 4; ++nn) PU[m][nn] = 0.0;
    const double G[4] = {0.0, 1.0, 1.0, gm.G3};
#pragma unroll
    for (int k = 1; k <= D; ++k) {
      double s0 = 0.0;
#pragma unroll
      for (int j = 1; j <= D; ++j) {
        const double d = so.DU[(k - 1) * 3 + (j - 1)][i];
        PU[k][j] = d;
        s0 += G[j] * in.u[j] * d;
      }
      PU[k][0] = s0 * in.igam;
    }
#pragma unroll
    for (int nn = 0; nn < 4; ++nn) {
      double s0 = 0.0;
#pragma unroll
      for (int k = 1; k <= 3; ++k) s0 -= in.v[k] * PU[k][nn];
      PU[0][nn] = s0;                                         /* + du^nn, added per trial */
    }
#pragma unroll
    for (int m = 0; m < 4; ++m)
#pragma unroll
      for (int nn = 0; nn < 4; ++nn) in.CDc[m][nn] = PU[m][nn];
    if (gm.hyper) {
      in.CDc[3][0] += gm.tau * in.u[3];          /* Gamma^0_{33} u^3 */
      in.CDc[0][3] += in.u[3] * in.itau;          /* Gamma^3_{03} u^3 */
      in.CDc[3][3] += in.gam * in.itau;           /* Gamma^3_{30} u^0 */
    }
#pragma unroll
    for (int nn = 0; nn < 4; ++nn) {
      double s0 = 0.0;
#pragma unroll
      for (int m = 0; m < 4; ++m) s0 += in.u[m] * in.CDc[m][nn];
      in.Duc[nn] = s0;
    }
  }
  in.thc = in.gam * (so.divv[i] + gm.Gamma_g);
#pragma unroll
  for (int k = 0; k < 3; ++k) in.FM[k] = (k < D) ? gm.sqrtg * (so.FP[k][i] - so.FB[k][i]) : 0.0;
#pragma unroll
  for (int q = 0; q < NQ; ++q) in.FKs[q] = gm.sqrtg * so.FK[q][i];
  in.uI = 0.0;
  if (rk.src) {
    /* source terms, Eq. 38 (:623), Eq. 42-44 (:645-649), Eq. 96 (:1003):
         d/dx0 [C u_i + pi~^0_i / gamma] += I_i / (gamma sigma),  d/dx0 [N_q + J~^0_q / gamma] += I_q / (gamma sigma),
         gamma sigma (T dS + mu_q dN_q)  += u_mu I^mu */
    const int64_t oid = rk.orig[a];
    const double igs = in.igam * in.isig;
#pragma unroll
    for (int m = 0; m < 4; ++m) {
      const double Im = (m <= D) ? rk.src[m * npad + oid] : 0.0;
      in.uI += in.ulo[m] * Im;
      if (m >= 1 && m <= D) in.FM[m - 1] += in.glo[m] * Im * igs;
    }
#pragma unroll
    for (int q = 0; q < NQ; ++q) in.FKs[q] -= rk.src[(4 + q) * npad + oid] * igs;
  }
  if (kp.diff) {
    /* tau_q sigma [...] = -J^i_q + sum_q' kappa_qq' nabla^<i> alpha_q',  nabla^<i> alpha = g^{ii} d_i alpha - u^i u^j d_j alpha */
    double udota[NQ];
#pragma unroll
    for (int r = 0; r < NQ; ++r) {
      double s0 = 0.0;
#pragma unroll
      for (int j = 1; j <= D; ++j) s0 += in.u[j] * so.DA[r * 3 + (j - 1)][i];
      udota[r] = s0;
    }
#pragma unroll
    for (int q = 0; q < NQ; ++q)
#pragma unroll
      for (int k = 1; k <= D; ++k) {
        double rhs = -in.sig * in.ds.Jt[q][k];
#pragma unroll
        for (int r = 0; r < NQ; ++r) rhs += in.kappa[q][r] * (in.gup[k] * so.DA[r * 3 + (k - 1)][i] - in.u[k] * udota[r]);
        in.rhsJ[q][k - 1] = rhs;
      }
  }

  /* residual at du = 0 and at the unit vectors -> D x D system of Eq. 95 */
  EomOut o;
#ifdef CCAKE_EOM_COMBINE
  EomOut oB[3];                /* the outputs of the homogeneous columns, combined with the solution below */
#endif
  double r0[3], M[3][3] = {{0.0, 0.0, 0.0}, {0.0, 0.0, 0.0}, {0.0, 0.0, 0.0}}, du[3] = {0.0, 0.0, 0.0};
#ifdef CCAKE_EOM_COMBINE
  eom_rates<D, 1>(kp, gm, in, du, o);
#pragma unroll
  for (int k = 0; k < D; ++k) r0[k] = o.res[k];
  eom_rates<D, 2>(kp, gm, in, du, oB[0]);
  eom_rates<D, 3>(kp, gm, in, du, oB[1]);
  if (D == 3) eom_rates<D, 4>(kp, gm, in, du, oB[2]);
#pragma unroll
  for (int c = 0; c < D; ++c)
#pragma unroll
    for (int k = 0; k < D; ++k) M[k][c] = oB[c].res[k];
#else
  eom_rates<D, 1>(kp, gm, in, du, o);
#pragma unroll
  for (int k = 0; k < D; ++k) r0[k] = o.res[k];
  /* columns of the matrix: the homogeneous part of the map at e_c, each a specialised (much shorter) evaluation */
  eom_rates<D, 2>(kp, gm, in, du, o);
#pragma unroll
  for (int k = 0; k < D; ++k) M[k][0] = o.res[k];
  eom_rates<D, 3>(kp, gm, in, du, o);
#pragma unroll
  for (int k = 0; k < D; ++k) M[k][1] = o.res[k];
  if (D == 3) {
    eom_rates<D, 4>(kp, gm, in, du, o);
#pragma unroll
    for (int k = 0; k < D; ++k) M[k][2] = o.res[k];
  }
#endif
  /* Gaussian elimination with partial pivoting */
  double b[3];
  bool ok = true;
#pragma unroll
  for (int k = 0; k < D; ++k) b[k] = -r0[k];
#pragma unroll
  for (int c = 0; c < D; ++c) {
    int piv = c;
#pragma unroll
    for (int r = c + 1; r < D; ++r) if (fabs(M[r][c]) > fabs(M[piv][c])) piv = r;
    if (M[piv][c] == 0.0 || !(fabs(M[piv][c]) < INFINITY)) { ok = false; break; }
    if (piv != c) {
#pragma unroll
      for (int k = 0; k < D; ++k) { const double t = M[c][k]; M[c][k] = M[piv][k]; M[piv][k] = t; }
      const double t = b[c]; b[c] = b[piv]; b[piv] = t;
    }
#pragma unroll
    for (int r = c + 1; r < D; ++r) {
      const double f = M[r][c] / M[c][c];
#pragma unroll
      for (int k = c; k < D; ++k) M[r][k] -= f * M[c][k];
      b[r] -= f * b[c];
    }
  }
  if (ok)
#pragma unroll
    for (int r = D - 1; r >= 0; --r) {
      double s0 = b[r];
#pragma unroll
      for (int k = r + 1; k < D; ++k) s0 -= M[r][k] * du[k];
      du[r] = s0 / M[r][r];
    }
  double sgsq = 0.0;
#ifdef CCAKE_EOM_COMBINE
  if (DIAG) {
    eom_rates<D, 0>(kp, gm, in, du, o, &sgsq);
  } else {
    /* the rates are affine in du: out(du) = out(0) + sum_c du_c * (homogeneous part at e_c) */
#pragma unroll
    for (int c = 0; c < D; ++c) {
      const double w = du[c];
      o.theta = fma(w, oB[c].theta, o.theta);
      o.dS = fma(w, oB[c].dS, o.dS);
      o.dBulk = fma(w, oB[c].dBulk, o.dBulk);
#pragma unroll
      for (int q = 0; q < NQ; ++q) {
        o.dN[q] = fma(w, oB[c].dN[q], o.dN[q]);
#pragma unroll
        for (int j = 1; j <= D; ++j) o.dJt[q][j] = fma(w, oB[c].dJt[q][j], o.dJt[q][j]);
      }
#pragma unroll
      for (int i = 1; i <= 3; ++i)
#pragma unroll
        for (int j = i; j <= 3; ++j) o.dpit[i][j] = fma(w, oB[c].dpit[i][j], o.dpit[i][j]);
    }
  }
#else
  eom_rates<D, 0>(kp, gm, in, du, o, DIAG ? &sgsq : nullptr);
#endif
  if (DIAG) {                                      /* applicability diagnostics, Eq. 58-61 (:797-805) */
    double pp = 0.0;
#pragma unroll
    for (int m = 0; m < 4; ++m)
#pragma unroll
      for (int n = 0; n < 4; ++n) { const double pv = in.sig * in.ds.pit[m][n]; pp += in.glo[m] * in.glo[n] * pv * pv; }
    rk.diag[0 * npad + i] = in.tau_pi * sqrt(fmax(sgsq, 0.0));
    rk.diag[1 * npad + i] = sqrt(fmax(pp, 0.0)) / in.p;
    rk.diag[2 * npad + i] = in.tau_Pi * o.theta;
    rk.diag[3 * npad + i] = fabs(in.ds.bulkt * in.sig) / in.p;
  }
  if ((!ok || !(o.dS == o.dS) || !(du[0] == du[0])) && (int64_t)rk.orig[a] < rk.n_own) atomicAdd(&status->n_bad, 1ULL);

  /* rates of the evolved set */
  double k_[NSTATE];
#pragma unroll
  for (int f = 0; f < NSTATE; ++f) k_[f] = 0.0;
#pragma unroll
  for (int j = 1; j <= D; ++j) { k_[CCAKE_R1 + j - 1] = in.u[j] * in.igam; k_[CCAKE_U1 + j - 1] = du[j - 1]; }
  k_[CCAKE_S] = o.dS;
#pragma unroll
  for (int q = 0; q < NQ; ++q) k_[CCAKE_NB + q] = o.dN[q];
  k_[CCAKE_BULK] = o.dBulk;
  k_[CCAKE_PI11] = o.dpit[1][1]; k_[CCAKE_PI12] = o.dpit[1][2]; k_[CCAKE_PI22] = o.dpit[2][2]; k_[CCAKE_PI33] = o.dpit[3][3];
  if (D == 3) { k_[CCAKE_PI13] = o.dpit[1][3]; k_[CCAKE_PI23] = o.dpit[2][3]; }
#pragma unroll
  for (int q = 0; q < NQ; ++q)
#pragma unroll
    for (int j = 1; j <= D; ++j) k_[CCAKE_JB1 + 3 * q + j - 1] = o.dJt[q][j];
  /* 2+1D hyperbolic: longitudinal work rate (DESIGN reading 14) */
  if (gm.hyper && D == 2) {
    const double Pi = in.ds.bulkt * in.sig;
    k_[CCAKE_WORK] = (Y[CCAKE_MASS * npad + a] / in.sst) * (in.p + Pi + gm.tau * gm.tau * in.sig * in.ds.pit[3][3]);
  }
  if (rk.theta_out) rk.theta_out[i] = o.theta;
  if (rk.Krate)
#pragma unroll
    for (int f = 0; f < NSTATE; ++f) if (f != CCAKE_MASS) rk.Krate[f * npad + a] = k_[f];
  if (rk.update) {
#pragma unroll
    for (int f = 0; f < NSTATE; ++f) {
      if (!(field_mask & (1u << f)) || f == CCAKE_MASS) continue;
      const double y0 = rk.Ybase[f * npad + a];
      double kk = k_[f];
      if (rk.acc_mode == 1) rk.Yacc[f * npad + a] = kk;
      else if (rk.acc_mode == 2) { rk.Yacc[f * npad + a] = rk.Yacc[f * npad + a] + rk.w_acc * kk; }
      else if (rk.acc_mode == 3) kk = rk.Yacc[f * npad + a] + kk;
      rk.Yout[f * npad + a] = y0 + rk.c_out * kk;
    }
    if (rk.Yout != rk.Ybase) rk.Yout[CCAKE_MASS * npad + a] = rk.Ybase[CCAKE_MASS * npad + a];
  }
}

}  // namespace ccake
