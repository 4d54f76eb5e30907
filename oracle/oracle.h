/*
 * oracle/oracle.h — C ABI of the CPU ORACLE.  TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * The oracle is a plain, slow, fp64 CPU restatement of one Runge-Kutta (sub)step of the CCAKE 2.0 SPH
 * fluid solver as PAPER.md states it (§5.6 SPH, §5.2 EoM, §5.3 transport, §5.1/App. A EoS) under the readings
 * listed in DESIGN.md.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may load it.  It shares NO code, header, table or constant generator with the CUDA library
 * (include/ccake.h, paper_2511_22852_b200/csrc); the numeric field ids below are restated, not included.
 *
 * All quantities are in fm units (hbar = c = 1): T, mu in fm^-1; s, n_q in fm^-3; e, p in fm^-4.
 * All buffers are HOST memory; the caller owns every buffer it passes.
 * Every call returns 0 or a negative code (ORACLE_E*); text via oracle_last_error().
 */
#ifndef CCAKE_ORACLE_H
#define CCAKE_ORACLE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

enum {
  ORACLE_OK = 0, ORACLE_EINVAL = -1, ORACLE_ENOMEM = -2, ORACLE_ESTATE = -4, ORACLE_ERANGE = -5
};

/* field ids: state (load + read) */
enum {
  OF_R1 = 0, OF_R2, OF_R3, OF_U1, OF_U2, OF_U3, OF_S, OF_NB, OF_NS, OF_NQ, OF_BULK,
  OF_PI11, OF_PI12, OF_PI13, OF_PI22, OF_PI23, OF_PI33,
  OF_JB1, OF_JB2, OF_JB3, OF_JS1, OF_JS2, OF_JS3, OF_JQ1, OF_JQ2, OF_JQ3,
  OF_MASS = 26, OF_WORK = 27, OF_NSTATE = 28,
  /* applicability diagnostics, Eq. 58-61 (:797-805): Kn_pi = tau_pi sqrt(sigma^{mn} sigma_{mn}),
     Re_pi^-1 = sqrt(pi^{mn} pi_{mn}) / p, Kn_Pi = tau_Pi theta, Re_Pi^-1 = |Pi| / p; read only */
  OF_KN_PI = 28, OF_RE_PI, OF_KN_BULK, OF_RE_BULK,
  /* derived, read only; evaluated at the current state */
  OF_SIGMA_STAR = 32, OF_S_DENS, OF_RHO_B, OF_RHO_S, OF_RHO_Q, OF_T, OF_MU_B, OF_MU_S, OF_MU_Q,
  OF_P = 41, OF_E, OF_CS2, OF_GAMMA, OF_NNB, OF_CELL, OF_THETA, OF_SIGMA, OF_S_STAR,
  OF_RHOSTAR_B = 50, OF_RHOSTAR_S, OF_RHOSTAR_Q, OF_WS, OF_DIVV,
  OF_FM1 = 55, OF_FM2, OF_FM3,   /* sqrt(-g) (FP_i - FB_i): right-hand side of the momentum equation */
  OF_FK_B = 58, OF_FK_S, OF_FK_Q, /* -sqrt(-g) FK_q: right-hand side of the charge equation           */
  /* OF_RATE + state id: d(state field)/dx0 at the current state */
  OF_RATE = 64,
  /* freeze-out surface element of PAPER.md §5.10, Eq. 145-148 (:1466-1482), per particle at the current state:
     d_mu eps (mu = 0..3), the outward unit normal n_mu = -d_mu eps / sqrt|d eps . d eps| and
     |d sigma| = m / (sigma |u^mu n_mu|); read only */
  OF_FO_DE0 = 96, OF_FO_DE1, OF_FO_DE2, OF_FO_DE3, OF_FO_N0, OF_FO_N1, OF_FO_N2, OF_FO_N3, OF_FO_DSIGMA
};

typedef struct oracle_params {
  int32_t dim;         /* 2 | 3 evolved spatial dimensions                                        */
  int32_t coords;      /* 0 Cartesian (t,x,y,z) | 1 hyperbolic (tau,x,y,eta_s)                    */
  int32_t integrator;  /* 2 RK2 midpoint | 4 classical RK4                                        */
  int32_t eom;         /* 0 ideal | 1 Israel-Stewart minimal (Eq. 49-51) | 2 DNMR shear+bulk      */
  int32_t flags;       /* bit0 shear, bit1 bulk, bit2 BSQ diffusion (ignored when eom == 0)       */
  int32_t eos_kind;    /* 0 closed-form conformal (c0,c2,c4) | 1 table                            */
  int32_t neighbour_mode; /* 0 cell list | 1 O(N^2) brute force                                   */
  int32_t reserved0;
  double h, x0_start, dx0;
  double eos_c0, eos_c2, eos_c4;
  double eta_over_s, tau_pi_coeff, tau_floor;
  double zeta_max, zeta_T_peak, zeta_width, tau_Pi_coeff;
  double kappa_over_T2[9];
  double tau_q_times_T[3];
  double dnmr_coeffs[8];
} oracle_params;

typedef struct oracle_ctx oracle_ctx;

int oracle_create(const oracle_params* p, oracle_ctx** out);
int oracle_destroy(oracle_ctx* c);
int oracle_load_particles(oracle_ctx* c, int64_t n, int32_t nfields, const int32_t* field_ids,
                          const double* const* cols);
int oracle_load_eos_table(oracle_ctx* c, const int32_t dims[4], const int32_t axis_kind[4],
                          const double* const axes[4], int32_t ncols, const int32_t* col_ids,
                          const double* data);
int oracle_step(oracle_ctx* c, int32_t nsteps);
int oracle_read_fields(oracle_ctx* c, int32_t nfields, const int32_t* field_ids, double* const* cols,
                       int64_t capacity);
int oracle_conserved_totals(oracle_ctx* c, double out[16]);
int oracle_read_neighbors(oracle_ctx* c, int64_t* counts, int64_t* offsets, int32_t* list, int64_t cap);
const char* oracle_last_error(const oracle_ctx* c);

/* oracle-only pins */
double oracle_kernel_W(int32_t D, double h, double r);
void oracle_kernel_gradW(int32_t D, double h, const double dr[3], double out[3]);
int oracle_eos_closed_form(const oracle_params* p, double s, const double n[3], double out[11]);
int oracle_eos_forward(const oracle_params* p, double T, const double mu[3], double out[5]);
int oracle_eos_table_lookup(oracle_ctx* c, double s, const double n[3], double out[11], int32_t* oob);

/* Offline inverter on a TABULATED forward EoS (PAPER.md :576-593; DESIGN reading 21): fdata holds (p, s, n_B, n_S, n_Q) at
 * the nodes of the (T, mu_B, mu_S, mu_Q) grid faxes (strictly increasing, fdims nodes each, last axis fastest).  For each
 * of the nt targets (s[a], n[q][a]): damped 4-D Newton on the quadrilinear interpolant; out[a*11 .. a*11+10] = T, mu_B,
 * mu_S, mu_Q, p, c_s^2, e, dw/ds, dw/dn_B, dw/dn_S, dw/dn_Q; flag[a] = 0 (found in the table) or 1 (the backup EoS,
 * the closed-form conformal one of *p, was used); iters (may be NULL) = Newton iterations taken. */
int oracle_invert_forward_table(const oracle_params* p, const int32_t fdims[4], const double* const faxes[4], const double* fdata,
                                int64_t nt, const double* s, const double* const n[3], double* out, int32_t* flag, int32_t* iters);

/* Source smearing of PAPER.md Eq. 35 (:521), the gather half of the dynamical initialisation: for every loaded
 * particle i,  j^mu_i = eta_norm / (dx0 sqrt(-g)) * sum over partons k with x0 - dx0 < t_k <= x0 of
 * p^mu_k W(r_i - r_k; h_source), W the cubic spline of Eq. 77 in the context's dimension, x0 the current time and
 * dx0 the step of the context.  p: 4 columns, r: 3 columns (dim used), t: formation times, np entries each;
 * j: 4 columns of n doubles (particle order).  The state is not modified. */
int oracle_smear_sources(oracle_ctx* c, int64_t np, const double* const p[4], const double* const r[3], const double* t,
                         double h_source, double eta_norm, double* const j[4]);

/* Source terms of the conservation equations, Eq. 38 (:623), Eq. 42-44 (:645-649), Eq. 96 (:1003):
 * nabla_mu T^{mu nu} = I^nu, nabla_mu N^mu_q = I_q.  I: 4 columns (contravariant I^mu per particle, e.g. the j^mu of
 * oracle_smear_sources), Iq: 3 columns; n doubles each; a NULL array or NULL column means zero.  They stay in force for
 * every evaluation until set again.  In the conservative per-particle form of Step 5:
 *   d/dx0 [ C u_i + pi~^0_i / gamma ] = sqrt(-g) (FP_i - FB_i) + I_i / (gamma sigma),       I_i = g_ii I^i
 *   d/dx0 [ N_q + J~^0_q / gamma ]     = -sqrt(-g) FK_q + I_q / (gamma sigma)
 *   gamma sigma (T dS + mu_q dN_q)     = u_mu I^mu - Pi theta + pi^mu_nu nabla_mu u^nu                          */
int oracle_set_sources(oracle_ctx* c, const double* const I[4], const double* const Iq[3]);

#ifdef __cplusplus
}
#endif
#endif
