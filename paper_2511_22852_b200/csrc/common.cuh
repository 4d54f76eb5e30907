/*
 * csrc/common.cuh — shared declarations of the CUDA library (product code; shares nothing with oracle/).
 *
 * Data layout in HBM (DESIGN.md §"Data layout"): structure of arrays, one fp64 array per field.
 *   - "store order": the state buffers Y0 / Ystage / Yacc hold CCAKE_NSTATE fields of N doubles each, field f at
 *     Y + f * Npad.  Store order is the cell-sorted order of the first substep of the current step; orig_id maps a
 *     store slot back to the caller's original index.
 *   - "sorted order": per-substep packed arrays (positions, smoothing payload, sums, thermodynamics, pair payload,
 *     gradient sums) in the order of the stable radix sort by cell; perm[i] = store slot of sorted slot i.
 */
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/ccake.h"

namespace ccake {

constexpr int NQ = 3;
constexpr int NSTATE = CCAKE_NSTATE;
constexpr double GRID_MARGIN = 1.0 + 1.0 / 1048576.0; /* traversal-grid edge = 2h (1 + 2^-20): rounding in the
                                                          cell index can never hide a pair with r^2 < (2h)^2 */

/* uniform traversal grid of one substep, written by the bbox kernel, read by every later kernel */
struct Grid {
  double xmin[3], xmax[3];
  double edge, inv_edge;
  int nc[3];
  int ncells;
  /* reported cell id (DESIGN reading 9): edge exactly 2h */
  double rep_inv_edge;
  long long rep_nc[3];
  /* sort key = (cell id << mb) | Hilbert index of the position inside the cell (mb bits) */
  int mb;
  /* FP32 culling: positions are stored relative to xmin; cutm = 2h + margin covering their rounding, cutm2 its
     square rounded up */
  double cutm;
  float cutm2;
};

/* Cell numbering ("snake"): rows of cells along x are numbered row = y' + nc[1] * z with y' running backwards in
   odd z-planes, and the cells of an odd row run backwards in x, so that consecutive cell ids are always face
   neighbours.  Together with the Hilbert index inside the cell (mirrored in x in odd rows) the sorted order is one
   continuous curve through the occupied space: every run of consecutive particles is spatially compact, also
   across cell and row ends.  Cells of one row are still contiguous in id, which is all the traversal needs. */
__host__ __device__ inline int snake_row(const Grid& g, int cy, int cz) {
  return ((cz & 1) ? g.nc[1] - 1 - cy : cy) + g.nc[1] * cz;
}
/* ids of the first and last cell of the physical x-range [x0, x1] of row `row` (first <= last) */
__host__ __device__ inline void snake_range(const Grid& g, int row, int x0, int x1, int& first, int& last) {
  const int base = g.nc[0] * row;
  if (row & 1) { first = base + g.nc[0] - 1 - x1; last = base + g.nc[0] - 1 - x0; }
  else { first = base + x0; last = base + x1; }
}
/* physical cell coordinates of a cell id */
__host__ __device__ inline void snake_decode(const Grid& g, uint32_t cid, int& cx, int& cy, int& cz) {
  const int row = (int)(cid / (uint32_t)g.nc[0]);
  const int xs = (int)(cid % (uint32_t)g.nc[0]);
  cz = row / g.nc[1];
  const int ys = row - cz * g.nc[1];
  cy = (cz & 1) ? g.nc[1] - 1 - ys : ys;
  cx = (row & 1) ? g.nc[0] - 1 - xs : xs;
}

/* geometry of a time slice: g = diag(1, -1, -1, -G3), G3 = tau^2 (hyperbolic) or 1 */
struct Geom {
  double G3, dG3, sqrtg, Gamma_g, tau;
  int hyper;
};

__host__ __device__ inline Geom make_geom(int coords, double x0) {
  Geom g;
  g.hyper = coords;
  g.tau = x0;
  if (coords == 1) { g.G3 = x0 * x0; g.dG3 = 2.0 * x0; g.sqrtg = x0; g.Gamma_g = 1.0 / x0; }
  else { g.G3 = 1.0; g.dG3 = 0.0; g.sqrtg = 1.0; g.Gamma_g = 0.0; }
  return g;
}

/* constant parameters handed to kernels by value */
struct KParams {
  int D, coords, eom, eos_kind;
  int shear, bulk, diff;
  double h, inv_h, cut2, sigma_d;   /* kernel normalisation sigma_D of Eq. 77 */
  /* folded constants of the cubic spline (Eq. 77, 79), set once on the host so that the pair kernels read them as
     constant-bank operands:  W = sigma_D (1 - 3/2 q^2 + 3/4 q^3) | sigma_D/4 (2-q)^3;
     (grad W)/dr = sigma_D/h^2 (9/4 q - 3) | -3/4 sigma_D/h (2-q)^2 / r */
  double w_a, w_b, w_c, g_a, g_b, g_c;
  double c0, c2, c4;
  double eta_over_s, tau_pi_coeff, tau_floor;
  double zeta_max, zeta_T_peak, zeta_width, tau_Pi_coeff;
  double kappa_over_T2[9], tau_q_times_T[3], dnmr[8];
};

/* EoS table descriptor (device pointers).  data: TB_STRIDE doubles per node, column id c at position c (absent columns 0),
   nodes in the caller's order (last axis fastest); col_of / ncols describe the caller's layout (table_pack_kernel).
   ax[0..3] are consecutive pieces of ONE array (ax[k + 1] = ax[k] + dims[k]). */
constexpr int TB_STRIDE = 12;
static_assert(TB_STRIDE >= CCAKE_NCOLS_MAX && TB_STRIDE % 2 == 0, "node record");
struct TableDev {
  int dims[4], kind[4], ncols;
  int col_of[CCAKE_NCOLS_MAX];
  const double* ax[4];
  const double* data;
};

/* sorted-order work arrays of one substep (all device pointers, N entries each unless noted) */
struct Sorted {
  /* a3 */
  uint32_t *key, *perm;              /* cell id, store slot */
  uint32_t* cell_start;              /* ncells + 1, monotone */
  /* pack: exact positions (SoA), FP32 positions relative to grid.xmin, AoS payload of the smoothing pass */
  double* x[3];
  float4* xf;
  double* rec_s;      /* [n][8]: x[3], m, S, N_B, N_S, N_Q */
  /* a4 */
  double *sigma_star, *s_star, *rho_star[NQ];
  uint32_t* nnb;
  /* a5 */
  double *gamma, *sigma, *s, *n[NQ];
  double *T, *mu[NQ], *p, *e, *cs2, *ws, *wq[NQ];
  double* rec_g;      /* [n][32]: AoS payload of the gradient pass: 8 blocks of 4 MMA operands, position in the 3 free slots (pair_mma.cuh) */
  /* a6 */
  double *FP[3], *FB[3], *FK[NQ], *DU[9], *DA[9], *divv;
  /* hit masks of the smoothing pass, reused by the gradient pass of the same substep (pair_mma.cuh):
     [pair block][tile number < mask_tiles][group of 8 homes] x 128 bit; NULL / 0 = no reuse */
  uint4* mask_cache;
  int mask_tiles;
  /* candidate lists of the pair blocks, written once per substep by cand_list_kernel and read by both passes:
     block b owns cand_list[b * cand_cap ...], cand_cnt[b] entries (0xffffffff: did not fit, the pass lists its
     candidates itself); NULL / 0 = not available */
  uint32_t *cand_list, *cand_cnt;
  int cand_cap;
  /* freeze-out element (NEXT-2): SPH gradient of eps, written by pair_kernel<EpsGradOp>; NULL until requested */
  double* fo_de[3];
};

/* device-side status counters */
struct Status {
  unsigned long long n_oob;      /* particles outside the EoS table in the latest thermo pass */
  unsigned long long n_bad;      /* singular solves / NaN since the last load                 */
  unsigned long long n_oob_total;   /* ... summed over every substep of every step since the last load    */
};

}  // namespace ccake
