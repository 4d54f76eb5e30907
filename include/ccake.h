/*
 * include/ccake.h — C ABI of libccake: the B200-native (sm_100a) SPH hot path of CCAKE 2.0.
 *
 * The library advances the SPH state  phi_a = { r^i, u^i, S = s/sigma, N_q = n_q/sigma, Pi/sigma, pi^{ij}/sigma,
 * J^i_q/sigma }  (Eq. 85 :954) of all particles by explicit Runge-Kutta steps of  d phi_a / dx0
 * (Eq. 87 :964).  One RK substep runs, in this order and entirely in CUDA kernels on the context's stream
 * (DESIGN.md §"Kernels"):
 *   a1 bounding box, a2 cell hash, a3 stable radix sort by cell + cell lists      (PAPER.md :1434, §5.9.1)
 *   a4 smoothing sums sigma*, s*, rho*_B, rho*_S, rho*_Q                          (Eq. 71-72 :877-882, Eq. 77 :910)
 *   a5 rest-frame densities (Eq. 68 :864), equation of state: 4-D table gather by quadrilinear interpolation
 *      (:583-593) or the closed-form conformal family (App. A :2115-2156), transport coefficients (§5.3)
 *   a6 pairwise gradient sums with dW_ab (Eq. 79 :920, Eq. 81-82 :934-938)
 *   a7 per-particle equations of motion reduced to a D x D solve (Eq. 87-104 :964-1041, Eq. 95 :988)
 *   a8 RK stage update;  a9 conserved totals (§5.6.5 :1049-1063) on request.
 *
 * Units: fm (hbar = c = 1): T, mu in fm^-1; s, n_q in fm^-3; e, p in fm^-4.  All arithmetic is fp64.
 *
 * Conventions common to every call
 *   - Returns CCAKE_OK (0) or a negative CCAKE_E* code; never throws, aborts or prints.  Text of the last error
 *     of a context: ccake_last_error().
 *   - Ownership: the caller owns every buffer it passes; the library copies on load and writes into caller
 *     buffers on read.  The context owns its device memory until ccake_destroy().
 *   - `memspace`: CCAKE_HOST (0) = host pointers, CCAKE_DEVICE (1) = device pointers on the context's device
 *     (e.g. torch.Tensor.data_ptr()).  Pointer ARRAYS (cols, axes, field_ids) are always host arrays.
 *   - Work is enqueued on the context's stream.  ccake_step() is asynchronous; calls that return data to the
 *     host synchronise the stream before returning.  One context per host thread.
 *   - There is no CPU fallback: without a usable CUDA device ccake_create() fails with CCAKE_ECUDA.
 */
#ifndef CCAKE_H
#define CCAKE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

enum { CCAKE_OK = 0, CCAKE_EINVAL = -1, CCAKE_ENOMEM = -2, CCAKE_ECUDA = -3, CCAKE_ESTATE = -4, CCAKE_ERANGE = -5 };
enum { CCAKE_HOST = 0, CCAKE_DEVICE = 1 };

/* Field ids.  State fields can be loaded and read; derived fields are read-only and are evaluated at the
 * current state (one evaluation of steps a1-a7 without an update). */
enum {
  CCAKE_R1 = 0, CCAKE_R2, CCAKE_R3,           /* position r^i (x, y, z | eta_s)                                */
  CCAKE_U1, CCAKE_U2, CCAKE_U3,               /* contravariant u^i; u^0 = gamma follows from u.u = 1           */
  CCAKE_S, CCAKE_NB, CCAKE_NS, CCAKE_NQ,      /* S = s/sigma, N_q = n_q/sigma (Eq. 84-86)                      */
  CCAKE_BULK,                                 /* Pi/sigma                                                      */
  CCAKE_PI11, CCAKE_PI12, CCAKE_PI13, CCAKE_PI22, CCAKE_PI23, CCAKE_PI33,   /* pi^{ij}/sigma                  */
  CCAKE_JB1, CCAKE_JB2, CCAKE_JB3, CCAKE_JS1, CCAKE_JS2, CCAKE_JS3, CCAKE_JQ1, CCAKE_JQ2, CCAKE_JQ3, /* J^i_q/sigma */
  CCAKE_MASS = 26,                            /* SPH weight m_b (default 1, Eq. 75 :898)                       */
  CCAKE_WORK = 27,                            /* accumulated longitudinal work (2+1D hyperbolic), starts at 0  */
  CCAKE_NSTATE = 28,
  /* applicability diagnostics of PAPER.md Eq. 58-61 (:797-805), read only, evaluated at the current state:
     Kn_pi = tau_pi sqrt(sigma^{mn} sigma_{mn}), Re_pi^-1 = sqrt(pi^{mn} pi_{mn}) / p, Kn_Pi = tau_Pi theta,
     Re_Pi^-1 = |Pi| / p */
  CCAKE_KN_PI = 28, CCAKE_RE_PI, CCAKE_KN_BULK, CCAKE_RE_BULK,
  CCAKE_SIGMA_STAR = 32, CCAKE_S_DENS, CCAKE_RHO_B, CCAKE_RHO_S, CCAKE_RHO_Q,  /* sigma*, rest-frame s, n_q   */
  CCAKE_T, CCAKE_MU_B, CCAKE_MU_S, CCAKE_MU_Q,
  CCAKE_P = 41, CCAKE_E, CCAKE_CS2, CCAKE_GAMMA, CCAKE_NNB, CCAKE_CELL, CCAKE_THETA, CCAKE_SIGMA, CCAKE_S_STAR,
  CCAKE_RHOSTAR_B = 50, CCAKE_RHOSTAR_S, CCAKE_RHOSTAR_Q, CCAKE_WS, CCAKE_DIVV,
  CCAKE_FM1 = 55, CCAKE_FM2, CCAKE_FM3,       /* right-hand side of the momentum equation, sqrt(-g)(FP_i - FB_i) */
  CCAKE_FK_B = 58, CCAKE_FK_S, CCAKE_FK_Q,    /* right-hand side of the charge equation, -sqrt(-g) FK_q         */
  CCAKE_RATE = 64,                            /* CCAKE_RATE + state id: d(state field)/dx0 at the current state */
  /* NEXT-2 of SURVEY.md §8(f): freeze-out surface element of PAPER.md §5.10, Eq. 145-148 (:1466-1482), per particle
     at the current state: d_mu eps (mu = 0..3; SPH n = +1 derivative in space, first law + rates in time), the
     outward unit normal n_mu = -d_mu eps / sqrt|d eps . d eps|, and |d sigma| = m / (sigma |u^mu n_mu|) */
  CCAKE_FO_DE0 = 96, CCAKE_FO_DE1, CCAKE_FO_DE2, CCAKE_FO_DE3, CCAKE_FO_N0, CCAKE_FO_N1, CCAKE_FO_N2, CCAKE_FO_N3,
  CCAKE_FO_DSIGMA
};

/* EoS table column ids (ccake_load_eos_table): T, mu_B, mu_S, mu_Q, p, c_s^2, e, dw/ds|_n, dw/dn_B, dw/dn_S, dw/dn_Q */
enum {
  CCAKE_COL_T = 0, CCAKE_COL_MUB, CCAKE_COL_MUS, CCAKE_COL_MUQ, CCAKE_COL_P, CCAKE_COL_CS2, CCAKE_COL_E,
  CCAKE_COL_WS, CCAKE_COL_WB, CCAKE_COL_WSQ, CCAKE_COL_WQ, CCAKE_NCOLS_MAX
};

/* Plain data, copied by ccake_create(). */
typedef struct ccake_params {
  int32_t dim;         /* 2 | 3 evolved spatial dimensions                                               */
  int32_t coords;      /* 0 Cartesian (t,x,y,z) | 1 hyperbolic (tau,x,y,eta_s), PAPER.md :488            */
  int32_t integrator;  /* 2 RK2 midpoint | 4 classical RK4 (the paper names no scheme; DESIGN reading 7) */
  int32_t eom;         /* 0 ideal | 1 Israel-Stewart minimal (Eq. 49-51 :676-680) | 2 DNMR shear+bulk (Eq. 52) */
  int32_t flags;       /* bit0 shear, bit1 bulk, bit2 BSQ diffusion (ignored when eom == 0)              */
  int32_t eos_kind;    /* 0 closed-form conformal p = c0 T^4 + c2 T^2 sum mu^2 + c4 sum mu^4 | 1 table   */
  int32_t device;      /* CUDA device ordinal                                                            */
  int32_t reserved0;
  void*   stream;      /* cudaStream_t to enqueue on, or NULL for the default stream                     */
  double  h;           /* smoothing length, support 2h (Eq. 77)                                          */
  double  x0_start;    /* initial time t or tau (> 0 for hyperbolic)                                     */
  double  dx0;         /* step size of one full RK step                                                  */
  double  eos_c0, eos_c2, eos_c4;
  double  eta_over_s, tau_pi_coeff, tau_floor;              /* tau_pi = max(coeff * eta / w, floor)      */
  double  zeta_max, zeta_T_peak, zeta_width, tau_Pi_coeff;  /* zeta/s = zeta_max W^2/(W^2 + (T-T_peak)^2) or
                                                               constant zeta_max when zeta_width <= 0;
                                                               tau_Pi = tau_Pi_coeff * tau_pi              */
  double  kappa_over_T2[9];   /* row-major 3x3 kappa_qq'/T^2 (:769, :779)                                */
  double  tau_q_times_T[3];   /* tau_q T (:781)                                                           */
  double  dnmr_coeffs[8];     /* delta_PiPi/tau_Pi, lambda_Pipi/tau_Pi, delta_pipi/tau_pi, tau_pipi/tau_pi,
                                 lambda_piPi, phi_omega (coefficient of the vorticity term), 2 unused     */
} ccake_params;

typedef struct ccake_ctx ccake_ctx;   /* opaque; owns all device memory */

/* Create a context on params->device.  EINVAL for out-of-range parameters, ECUDA when the device or the
 * kernels (sm_100a) are unusable. */
int ccake_create(const ccake_params* p, ccake_ctx** out);
int ccake_destroy(ccake_ctx* c);

/* Load n particles.  cols[k] (n doubles, `memspace`) holds state field field_ids[k]; fields not given are 0
 * (MASS: 1).  Fields of switched-off sectors (and the third components when dim == 2) are ignored.  Resets the
 * time to x0_start.  Particle index = position in these arrays ("original order"). */
int ccake_load_particles(ccake_ctx* c, int64_t n, int32_t nfields, const int32_t* field_ids,
                         const double* const* cols, int32_t memspace);

/* The same in two halves, for a loop over independent particle sets (events): ccake_stage_particles starts copying the
 * HOST columns (pinned, for the copies to be asynchronous; they must stay untouched until ccake_load_staged has been
 * called) into a staging arena on a copy stream of its own and returns at once — the copies overlap the steps of the
 * resident set and the read-back of ccake_read_fields_async.  ccake_load_staged installs the staged set exactly as
 * ccake_load_particles would: device-side copies on the context's stream that wait, on the device, for the staged
 * columns; when the particle count equals the resident one it does not wait on the host at all.  One set can be staged
 * at a time: staging again before ccake_load_staged replaces it.  ESTATE: ccake_load_staged with nothing staged. */
int ccake_stage_particles(ccake_ctx* c, int64_t n, int32_t nfields, const int32_t* field_ids, const double* const* cols);
int ccake_load_staged(ccake_ctx* c);

/* Load the offline-inverted EoS table (PAPER.md :583-593).  Axis 0 is s; axes 1..3 are B, S, Q, each either the
 * density n_q (axis_kind 0) or the ratio n_q / s (axis_kind 1).  axes[k] = dims[k] strictly increasing node
 * values (any spacing, e.g. the paper's log-decade pattern).  data is row-major [d0][d1][d2][d3][ncols] with
 * column k holding quantity col_ids[k]; columns T..WS are required, WB..WQ when diffusion is on.  Lookup is
 * quadrilinear; coordinates outside the table are clamped and counted (totals[11]). */
int ccake_load_eos_table(ccake_ctx* c, const int32_t dims[4], const int32_t axis_kind[4],
                         const double* const axes[4], int32_t ncols, const int32_t* col_ids,
                         const double* data, int32_t memspace);

/* NEXT-1 of SURVEY.md §8(f): the offline inversion of the equation of state (PAPER.md :576-593, App. A
 * :2115-2156) done on the device, for the analytic conformal BSQ family of params
 * (p = c0 T^4 + c2 T^2 sum_q mu_q^2 + c4 sum_q mu_q^4).  For every node of the (s, B, S, Q) grid described by
 * dims / axis_kind / axes (same meaning as in ccake_load_eos_table; `memspace` says where axes[k] and out live) it
 * solves (T, mu_q) from (s, n_q) — the cubic of Eq. A.13-A.14 for mu_q(T) inside a bisection in T on the monotone
 * s(T, mu(T)) — evaluates p, e = 3p, c_s^2 = 1/3, dw/ds and dw/dn_q there, and installs the result as the
 * context's table exactly as ccake_load_eos_table would.  out may be NULL; otherwise it receives the table,
 * [d0][d1][d2][d3][ncols] doubles.  A tabulated equation of state goes through ccake_invert_forward_table. */
int ccake_invert_eos_table(ccake_ctx* c, const int32_t dims[4], const int32_t axis_kind[4],
                           const double* const axes[4], int32_t ncols, const int32_t* col_ids, double* out,
                           int32_t memspace);

/* Rest of NEXT-1: the offline inverter on a TABULATED forward EoS (PAPER.md :576-593, footnote :585; DESIGN reading 21).
 * fdata holds (p, s, n_B, n_S, n_Q) — 5 doubles per node — on the (T, mu_B, mu_S, mu_Q) grid faxes (fdims nodes per
 * axis, strictly increasing, any spacing; row-major, last axis fastest).  For every node (s*, n*_q) of the target grid
 * dims / axis_kind / axes (as in ccake_load_eos_table) one device thread solves interp(T, mu) = (s*, n*) by damped
 * Newton on the quadrilinear interpolant — start: mu = 0, T by bisection on s; at most 40 iterations, converged at
 * max |residual| <= 1e-13 s*; step halving until the residual decreases — and writes T, mu_q, p = interp, e = T s* - p +
 * mu_q n*_q, dw/ds, dw/dn_q and c_s^2 from the interpolant's Jacobian.  A node the root-finder does not reach takes the
 * backup EoS (:572): the closed-form conformal family of params, flag 1.  The result is installed as the context's
 * table; out ([d0][d1][d2][d3][ncols] doubles), flags (one int32 per node: 0 table, 1 backup) may be NULL; n_backup
 * (host, may be NULL) receives the number of flagged nodes.  faxes[k], fdata, axes[k], out, flags live in `memspace`. */
int ccake_invert_forward_table(ccake_ctx* c, const int32_t fdims[4], const double* const faxes[4], const double* fdata,
                               const int32_t dims[4], const int32_t axis_kind[4], const double* const axes[4], int32_t ncols,
                               const int32_t* col_ids, double* out, int32_t* flags, int64_t* n_backup, int32_t memspace);

/* NEXT-3 (part) of SURVEY.md §8(f): the source smearing of PAPER.md Eq. 35 (:521), the gather half of the dynamical
 * initialisation.  For every loaded particle i, at the context's current time x0 and step dx0,
 *   j^mu_i = eta_norm / (dx0 sqrt(-g)) * sum over partons k with x0 - dx0 < t[k] <= x0 of p[mu][k] W(r_i - r[.][k]; h_source),
 * W the cubic spline of Eq. 77 in the context's dimension (2 h_source cut-off), sqrt(-g) = tau (hyperbolic) or 1.
 * p: 4 columns, r: 3 columns (the first `dim` are used), t: formation times — npartons doubles each; j: 4 columns of
 * n doubles in the caller's particle order; all in `memspace`.  Every parton is tested against every particle (no
 * spatial index: parton counts per step are thousands).  The state is not modified; ccake_set_sources feeds j^mu into
 * the equations of motion. */
int ccake_smear_sources(ccake_ctx* c, int64_t npartons, const double* const p[4], const double* const r[3],
                        const double* t, double h_source, double eta_norm, double* const j[4], int32_t memspace);

/* The same smearing for callers that must not allocate (a region under CUDA graph capture, a tight serving loop, a harness
 * that forbids cudaMalloc): ccake_smear_sources allocates and frees two device buffers per call, this entry point calls no
 * cudaMalloc, cudaFree or allocating library routine.  Its scratch memory — the packed parton array — is a fixed array in
 * the library's device image: 8 x CCAKE_SMEAR_NOALLOC_MAX doubles = 1 MiB, held by every GPU that loads the library until
 * the process exits.  EINVAL, with ccake_last_error naming the limit, when npartons > CCAKE_SMEAR_NOALLOC_MAX.
 * p, r, t, j as in ccake_smear_sources but DEVICE memory only (the caller owns inputs and outputs; j[m] has n doubles and
 * is overwritten for every particle; with npartons == 0 the input columns may be NULL and j becomes 0).  Asynchronous on the context's stream: j is valid after ccake_synchronize (or in
 * stream order).  The result is the one ccake_smear_sources gives (same arithmetic in the same order).
 * The scratch array is shared by every call on a device — all contexts, all streams — and keeps the last call's partons:
 * each call overwrites the entries it reads (nothing has to be cleared), and two calls that overlap on the GPU (different
 * streams / contexts of one device) race; calls on one stream are ordered and safe.  The context must have been created
 * and loaded beforehand (those calls allocate).  ESTATE before a load. */
#define CCAKE_SMEAR_NOALLOC_MAX 16384
int ccake_smear_sources_noalloc(ccake_ctx* c, int64_t npartons, const double* const p[4], const double* const r[3],
                                const double* t, double h_source, double eta_norm, double* const j[4]);

/* Rest of NEXT-3: source terms of the conservation equations, Eq. 38 (:623) nabla_mu T^{mu nu} = I^nu,
 * nabla_mu N^mu_q = I_q, as they enter Eq. 42-44 (:645-649) and the entropy equation Eq. 96 (:1003).  I: 4 columns, the
 * contravariant I^mu per particle (for instance the j^mu of ccake_smear_sources; I[3] is ignored when dim == 2); Iq: 3
 * columns I_B, I_S, I_Q; n doubles each in the caller's particle order, in `memspace`.  A NULL array or column is zero;
 * both NULL switches the sources off.  The values are copied and stay in force for every substep of every following
 * step until set again; ccake_load_particles clears them.  In the per-particle form the kernels solve (DESIGN reading 4):
 *   d/dx0 [C u_i + pi~^0_i / gamma] = sqrt(-g) (FP_i - FB_i) + I_i / (gamma sigma),   I_i = g_ii I^i,
 *   d/dx0 [N_q + J~^0_q / gamma]     = -sqrt(-g) FK_q + I_q / (gamma sigma),
 *   gamma sigma (T dS + mu_q dN_q)   = u_mu I^mu - Pi theta + pi^mu_nu nabla_mu u^nu.
 * ESTATE before a load. */
int ccake_set_sources(ccake_ctx* c, const double* const I[4], const double* const Iq[3], int32_t memspace);

/* ---- Slab decomposition of ONE event over several contexts (not in the paper, which runs one
 * event per device).  A slab context owns the particles with lo <= r[axis] < hi (lo = -1e300 / hi = +1e300: no neighbour on
 * that side) and carries ghost copies of the neighbours' particles within halo_width of its faces.  halo_width must cover
 * two kernel supports plus the drift of a step (>= 4h + 2 dx0): then ONE exchange of particle states per substep suffices —
 * the context recomputes smoothing sums and thermodynamics of its ghosts, so the gradient sums of every owned particle see
 * complete neighbours.  The caller moves the messages between contexts (device copy, or NCCL send/recv between ranks):
 *   per step:  for both sides: export_halo(k=0) -> [transport] -> neighbour.import_ghosts(k=0)     (low side first)
 *              substep(0);  for k = 1 .. nsub-1:  export_halo(k) -> import_ghosts(k);  substep(k)
 *              for both sides: export_migrants -> [transport] -> neighbour.import_migrants;  commit
 * Messages are DEVICE buffers of the caller: 29 rows of buf_cap doubles, row f < 28 = state field f, row 28 = the global
 * particle id; entry i of every row is particle i of the message, in the sender's store order (deterministic).  Load
 * indices of a slab context: owned particles 0 .. n_own-1 (after a commit: the stayers in sorted order, then the
 * arrivals), ghosts behind them; ccake_read_fields returns all of them in that order, ccake_slab_gids their global ids,
 * ccake_conserved_totals sums over the owned particles only (the caller adds the slabs).  The reported CELL id is relative
 * to the slab's own bounding box.  A slab context cannot take ccake_step; ESTATE for slab calls on other contexts. */
int ccake_slab_load(ccake_ctx* c, int64_t n_own, int64_t capacity, int32_t nfields, const int32_t* field_ids,
                    const double* const* cols, const uint32_t* gids, int32_t axis, double lo, double hi, double halo_width,
                    int32_t memspace);
/* side: 0 = the face at lo, 1 = the face at hi.  k = substep about to be evaluated: k = 0 selects the owned particles
 * within halo_width of the face from the state at the start of the step; k > 0 packs the same particles again from the
 * stage state.  *count = particles in the message (ENOMEM if it exceeds buf_cap; synchronises the stream). */
int ccake_slab_export_halo(ccake_ctx* c, int32_t side, int32_t k, double* buf, int64_t buf_cap, int64_t* count);
/* k = 0: the message becomes the ghosts of this step on that side (the ghosts of the previous step went with the commit);
 * k > 0: the stage state of those ghosts is overwritten (same count, same order). */
int ccake_slab_import_ghosts(ccake_ctx* c, int32_t side, int32_t k, const double* buf, int64_t buf_cap, int64_t count);
/* Substep k (0 .. 1 for RK2, 0 .. 3 for RK4) of one RK step over owned particles and ghosts; the last one advances the time. */
int ccake_slab_substep(ccake_ctx* c, int32_t k);
/* NARROW halos (halo_width >= 2h + 2 dx0 only): the ghosts' own smoothing sums are incomplete, so their gradient records
 * (32 doubles each: the payload columns of a6 and the position) come from their owners between a5 and a6:
 *   ccake_slab_substep_part(k, 1)  [a1-a5]  ->  export_records -> [transport] -> neighbour.import_records  ->
 *   ccake_slab_substep_part(k, 2)  [a6-a8]
 * Record messages have 32 rows of buf_cap doubles, entry i = the i-th particle of this step's halo message of that side. */
int ccake_slab_substep_part(ccake_ctx* c, int32_t k, int32_t part);
int ccake_slab_export_records(ccake_ctx* c, int32_t side, double* buf, int64_t buf_cap, int64_t* count);
int ccake_slab_import_records(ccake_ctx* c, int32_t side, const double* buf, int64_t buf_cap, int64_t count);
/* After the last substep: the owned particles that left [lo, hi) through `side`, as a message. */
int ccake_slab_export_migrants(ccake_ctx* c, int32_t side, double* buf, int64_t buf_cap, int64_t* count);
int ccake_slab_import_migrants(ccake_ctx* c, int32_t side, const double* buf, int64_t buf_cap, int64_t count);
/* Rebuild the owned set: stayers (store order) + arrivals from the low side + arrivals from the high side; ghosts dropped.
 * The load indices change, so sources set with ccake_set_sources are switched off and have to be set again. */
int ccake_slab_commit(ccake_ctx* c, int64_t* n_own_new);
/* out = { n_own, ghosts from the low side, ghosts from the high side, capacity } */
int ccake_slab_info(ccake_ctx* c, int64_t out[4]);
/* Global ids by load index, n_own + ghosts entries. */
int ccake_slab_gids(ccake_ctx* c, uint32_t* out, int64_t capacity, int32_t memspace);

/* Enqueue nsteps full RK steps (each 2 or 4 substeps a1-a8).  Asynchronous.  ESTATE before a load or on a slab context.
 * On a stream other than the legacy default stream the launch sequence of a step is captured once as a CUDA graph (the
 * current time lives in device memory, so the kernel arguments do not change from step to step) and replayed; the results
 * are bit-identical to launching the kernels one by one (environment CCAKE_NO_GRAPH=1 forces the latter, as does
 * ccake_enable_timing). */
int ccake_step(ccake_ctx* c, int32_t nsteps);

/* Wait for the stream.  ERANGE when, since the last load, a particle left the EoS table, a per-particle solve
 * was singular or a field became NaN (the state stays readable); ECUDA on a device fault. */
int ccake_synchronize(ccake_ctx* c);

/* Read fields in ORIGINAL particle order into cols[k] (capacity doubles each, capacity >= n). */
int ccake_read_fields(ccake_ctx* c, int32_t nfields, const int32_t* field_ids, double* const* cols,
                      int64_t capacity, int32_t memspace);

/* The same into HOST buffers without waiting for them: the fields are gathered into a device arena on the context's stream
 * and copied out on a second stream, so the copies overlap whatever the caller enqueues next (the next load and step of a
 * double-buffered loop).  The buffers (pinned, for the copies to be asynchronous) are valid after ccake_read_fields_wait;
 * a second asynchronous read waits on the device, not on the host, for the first one's copies. */
int ccake_read_fields_async(ccake_ctx* c, int32_t nfields, const int32_t* field_ids, double* const* cols, int64_t capacity);
int ccake_read_fields_wait(ccake_ctx* c);

/* out (host) = { x0, E, P_1, P_2, P_3, S_tot, N_B, N_S, N_Q, sum m, work, n_out_of_table, max |trace pi|,
 *                n_bad, sum_a N_nb(a), n_out_of_table_total } at the current state (DESIGN.md §"Totals").
 * n_out_of_table counts the particles clamped to the EoS table in the evaluation at the current state;
 * n_out_of_table_total sums that count over every substep of every step since the last load. */
int ccake_conserved_totals(ccake_ctx* c, double out[16]);

/* Test hook: neighbour sets {b != a : r_ab^2 < (2h)^2} of the current state, ORIGINAL indices, ascending per
 * particle, CSR.  counts (n), offsets (n+1, may be NULL), list (cap entries, may be NULL to query counts);
 * all host pointers. */
int ccake_read_neighbors(ccake_ctx* c, int64_t* counts, int64_t* offsets, int32_t* list, int64_t cap);

/* Test hook for sizes where lists do not fit: per particle (original order) the order-free hash
 * sum_b mix64(b) mod 2^64 over its neighbour set, mix64 = the splitmix64 finaliser of (b + 1).  Host pointer.
 * The sets are the ones the smoothing pass itself used: the hash is accumulated by a test instantiation of the pair
 * kernel (same candidate lists, tiles, culling and exact test), not by a separate walk. */
int ccake_neighbor_hash(ccake_ctx* c, uint64_t* out, int64_t capacity);

/* Measurement hook: average device time in ms of each kernel group over the substeps run since the last
 * call (out[0..7] = bbox+hash+sort, pack, smoothing, thermo/EoS, gradient, EoM+update, totals, substeps). */
int ccake_kernel_times(ccake_ctx* c, double out[8]);
int ccake_enable_timing(ccake_ctx* c, int32_t on);

/* Measurement hook: *out = number of CUDA kernels this context enqueued since the previous call (host counter,
 * no synchronisation); the counter is then reset. */
int ccake_launch_count(ccake_ctx* c, int64_t* out);

/* Measurement hook: the FP64 rate of the device, TFLOP/s (2 flop per fused multiply-add), from chains of independent
 * fma.rn.f64 on every SM, best of 5 launches timed with CUDA events on the default stream.  bench.py divides the
 * pair passes' achieved flop rate by this number.  Needs no context. */
int ccake_measure_fp64_peak(int32_t device, double* tflops);

const char* ccake_last_error(const ccake_ctx* c);

/* Test knobs (environment, read by ccake_load_particles): CCAKE_CAND_CAP = entries per pair block of the candidate
 * lists (0: none — every block lists its candidates inside the pass), CCAKE_MASK_TILES = tiles per block whose hit
 * masks the smoothing pass keeps for the gradient pass (0: none).  They force the paths a production run takes only
 * when a block's neighbourhood outgrows its list or when device memory is short. */

#ifdef __cplusplus
}
#endif
#endif
