/*
 * csrc/pair_mma.cuh — steps a4 (smoothing sums) and a6 (gradient sums): the two neighbour passes.
 *
 *   a4  sigma*_a = sum_b m_b W_ab,  s*_a = sum_b m_b S_b W_ab,  rho*_{q,a} = sum_b m_b N_{q,b} W_ab
 *       (Eq. 71-72 :877-882), b over r_ab^2 < (2h)^2 including b = a; W = cubic spline (Eq. 77 :910).
 *   a6  n = -1 and n = +1 SPH derivatives (Eq. 81-82 :934-938; DESIGN reading 3) with dW_ab of Eq. 79 :920.
 *
 * Design.  With ~800 neighbours per particle these passes are bound by the FP64 pipe of the SM
 * (measured: 36.9 TFLOP/s with DFMA, 37.1 TFLOP/s with DMMA, and no more than that with both — one pipe).  Every
 * sum of both passes has the form
 *       C[a][t] = sum_b  w_j(a, b) * Y_t(b)          (a: home particle, b: neighbour, t: payload column)
 * with a pair weight w_j (m_b W_ab, or the component j of m_b grad W_ab) that takes ~25-30 FP64 instructions and a
 * payload column Y_t that is a property of b alone: a small dense contraction over b.  The kernel therefore runs
 * the geometry on the vector FP64 units — one (home, candidate) pair per lane — and the accumulation as FP64
 * tensor-core MMAs (mma.sync.m8n8k4.f64: 8 homes x 4 candidates x 8 payload columns, 512 flop per instruction):
 * the same FP64 work on the same pipe, but one issue slot instead of 42 FMAs per pair and 2 accumulator registers
 * per (tile, direction) instead of 62 per home particle, so the pipe is kept busy by 16 resident warps without
 * register pressure.  The fragment layout makes this natural: lane l holds A[row l/4][col l%4] = w_j(home l/4,
 * candidate l%4), B[row l%4][col l/4] = column l/4 of candidate l%4, and the two accumulators of home l/4.
 *
 *   - The store is sorted along one space-filling curve (snake over the cells, Hilbert index inside a cell;
 *     grid_sort.cuh), so 8 consecutive particles ("group") are a compact cluster; a warp owns PM_GPW groups, a
 *     block BH = 256 consecutive home particles.
 *   - Candidates of a block come from cand_list_kernel (once per substep, global memory, both passes) or, for a
 *     block whose list does not fit there, from a list built inside the pass (interleaved sweeps).  Their AoS
 *     payload records are copied with cp.async, HALF_B at a time and taken with a stride through the list, into a
 *     ring of NSLOT tiles (2 in the gradient pass, 6 in the smoothing pass) in shared memory (component-major, one-unit skew) whose arrival is tracked by one
 *     mbarrier per slot; there is no block barrier per tile.
 *   - Per tile and group the warp tests the HALF_B candidates against the FP32 box of the group's 8 homes (ballots)
 *     and compacts the survivors into a FIFO of byte offsets; quads of 4 candidates are taken from it.  Leftovers (< 4)
 *     form a partial quad (smoothing pass) or are copied into carry columns behind the ring and lead the next tile's
 *     FIFO (passes that read cached masks).
 *   - The neighbour decision is the exact FP64 test r2 = (dx*dx + dy*dy) + dz*dz < (2h)^2 with round-to-nearest
 *     multiplies and adds and no FMA contraction (DESIGN reading 8), per pair; a miss enters the MMA with weight
 *     exactly 0.  The smoothing pass records which candidates hit at least one home of the group and stores that
 *     exact union as the group's hit mask; the gradient pass of the same substep (same list, same tiles) reads it
 *     back instead of culling again, so 71 % of its evaluations are true neighbours on a regular lattice.
 *   - 1/r comes from MUFU.RSQ64H + one third-order step (1 ulp); the order of b is fixed by the list, the tile
 *     stride and the FIFO, so results are reproducible run to run (no atomics).
 */
#pragma once
#include <type_traits>

#include "common.cuh"

namespace ccake {

#ifndef CCAKE_PM_CARRY
#define CCAKE_PM_CARRY 1                     /* passes that read cached masks carry the < 4 left-over candidates of a tile over */
#endif
#ifndef CCAKE_CL_LBK
#define CCAKE_CL_LBK 4                       /* candidates a thread of cand_list_kernel tests per step */
#endif
#ifndef CCAKE_PM_WARPS
#define CCAKE_PM_WARPS 16
#endif
#ifndef CCAKE_PM_GPW
#define CCAKE_PM_GPW 1
#endif
constexpr int PM_WARPS = CCAKE_PM_WARPS;     /* warps per block                                  */
constexpr int PM_GPW = CCAKE_PM_GPW;         /* groups of 8 home particles per warp              */
constexpr int PT = 32 * PM_WARPS;            /* threads per block                                */
constexpr int NGRP = PM_WARPS * PM_GPW;      /* groups per block                                 */
constexpr int BH = 8 * NGRP;                 /* home particles per block                         */
#ifndef CCAKE_PM_TILE
#define CCAKE_PM_TILE 128
#endif
#ifndef CCAKE_PM_MINB
#define CCAKE_PM_MINB 2
#endif
constexpr int HALF_B = CCAKE_PM_TILE;        /* candidates per tile (a multiple of 32, at most 128) */
constexpr int PM_MINB = CCAKE_PM_MINB;       /* resident blocks per SM the register budget is set for */
constexpr int NR32 = HALF_B / 32;            /* candidates a lane tests per tile and group       */
#ifndef CCAKE_PM_NSLOT
#define CCAKE_PM_NSLOT 2
#endif
#ifndef CCAKE_PM_NSLOT_S
#define CCAKE_PM_NSLOT_S 6                   /* measured on C4 with tiles of 128: 4 / 5 / 6 / 7 / 8 slots -> 7.81 / 7.66 / 7.64 / 7.65 / 7.76 ms */
#endif
constexpr int NSLOT_G = CCAKE_PM_NSLOT;      /* tiles resident in shared memory: the current one and those in flight (Op::NSLOT) */
constexpr int NSLOT_S = CCAKE_PM_NSLOT_S;    /* ... of the smoothing pass, whose records are a quarter of the gradient pass's */
constexpr int RPW = HALF_B / PM_WARPS;       /* records of a tile each warp copies               */
#ifndef CCAKE_LCAP
#define CCAKE_LCAP 1536
#endif
constexpr int LCAP = CCAKE_LCAP;             /* block candidate list in shared memory (a multiple of HALF_B) */
constexpr int LB = 2;                        /* candidates per thread and listing step           */
constexpr int MAXROW = 32;                   /* rows of cells per listing batch                  */
#ifndef CCAKE_CAND_CAP
#define CCAKE_CAND_CAP 16384
#endif
constexpr int CAND_CAP = CCAKE_CAND_CAP;     /* default entries per pair block in the global candidate lists */
#ifndef CCAKE_MASK_TILES
#define CCAKE_MASK_TILES 96
#endif
constexpr int MASK_TILES = CCAKE_MASK_TILES; /* default tiles per block whose hit masks the smoothing pass keeps */
static_assert(HALF_B % 32 == 0 && HALF_B <= 128 && HALF_B % PM_WARPS == 0 && RPW <= 32 && LCAP % HALF_B == 0 && BH <= 1024, "tile layout");

__device__ __forceinline__ double dist2_exact(double dx, double dy, double dz, int D) {
  double r2 = __dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy));
  if (D == 3) r2 = __dadd_rn(r2, __dmul_rn(dz, dz));
  return r2;
}

/* squared FP32 distance from a point to a box (0 inside) */
template <int D>
__device__ __forceinline__ float box_dist2(const float4 p, const float* lo, const float* hi) {
  const float dx = fmaxf(fmaxf(lo[0] - p.x, p.x - hi[0]), 0.f);
  const float dy = fmaxf(fmaxf(lo[1] - p.y, p.y - hi[1]), 0.f);
  float d2 = dx * dx + dy * dy;
  if (D == 3) {
    const float dz = fmaxf(fmaxf(lo[2] - p.z, p.z - hi[2]), 0.f);
    d2 += dz * dz;
  }
  return d2;
}

__device__ __forceinline__ float warp_minf(float v) {
  for (int o = 16; o > 0; o >>= 1) v = fminf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
__device__ __forceinline__ float warp_maxf(float v) {
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

/* D[8x8] += A[8x4] B[4x8] in FP64 on the tensor cores.  Lane l: a = A[l/4][l%4], b = B[l%4][l/4],
   (c0, c1) = D[l/4][2 (l%4) + {0, 1}]. */
__device__ __forceinline__ void dmma_m8n8k4(double& c0, double& c1, double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

/* what both passes need of one (home, b) pair: separation, exact neighbour decision, q = r/h, 1/r */
template <int D>
struct PairGeom {
  double dr[3], q, rinv;
  bool hit;
  /* q < 1 decided on the high word (q >= 0): one integer compare instead of an FP64 one.  At q = 1 exactly both
     branches of the spline agree, so taking the outer one there is the same function. */
  __device__ __forceinline__ bool inner() const { return __double2hiint(q) < 0x3ff00000; }
  __device__ __forceinline__ void set(const KParams& kp, const double* xa, double xb, double yb, double zb, bool act) {
    dr[0] = xa[0] - xb;
    dr[1] = xa[1] - yb;
    dr[2] = (D == 3) ? xa[2] - zb : 0.0;
    const double r2 = dist2_exact(dr[0], dr[1], dr[2], D);
    hit = act && (r2 < kp.cut2);
    /* 1/sqrt: MUFU.RSQ64H seed (it reads the high word only, ~20 bits) and one third-order step
       y = y0 + y0 e (1/2 + 3/8 e), e = 1 - x y0^2 (error <= 1 ulp).  The seed is taken at max(high word, smallest
       normal) so that r2 = 0 — the home particle itself — gives a finite 1/r (then e = 1, q = r2 * rinv = 0, and
       the q <= 1 branches do not use 1/r); no branch to a slow path for denormal / infinite arguments, which
       cannot occur for a pair inside the cut-off. */
    double y0;
    const double xs = __hiloint2double(max(__double2hiint(r2), 0x00100000), 0);
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y0) : "d"(xs));
    const double e = fma(r2, -(y0 * y0), 1.0);
    const double pp = fma(e, 0.375, 0.5);
    rinv = fma(pp, y0 * e, y0);
    q = (r2 * rinv) * kp.inv_h;
  }
};

/* An operator describes one pass:
     NREC         doubles per staged record (even); elements 0, 1, 2 are the position (z = 0 in 2-D); every payload element
                  is already multiplied by the SPH weight m_b of its particle
     GIDMAJOR     the record stores the 4 operands of MMA column n contiguously at double 4 + 4 n (gradient pass); otherwise
                  column n of tile T for weight j is element elem(T, j, n) (one 8-byte load each)
     NJ           pair weights per (home, b): 1 (W) or D (the components of grad W)
     NT           MMA column tiles: the pass accumulates NT * NJ matrices of 8 homes x 8 columns
     elem(T,j,n)  record element that is column n of tile T for weight j; ELEM_NONE = unused column
     weights()    the NJ pair weights of one pair, 0 for a miss
     finish()     combines the 8 * NT * NJ sums of one home particle and writes the outputs                     */
constexpr int ELEM_NONE = -2;

/* ------------------------------------------------------------------------------------------ a4 operator ---- */
/* record: x[3], m, m S, m N_B, m N_S, m N_Q  (z = 0 in 2-D).  HASH: test instantiation that also sums
   mix64(original id of b + 1) over the neighbour set the kernel actually used (ccake_neighbor_hash). */
template <int D_, bool HASH_ = false>
struct SmoothOp {
  static constexpr int D = D_;
  static constexpr bool HASH = HASH_;
  static constexpr bool COUNT = true, GIDMAJOR = false, CARRY = false;
  static constexpr int NREC = 8, NJ = 1, NT = 1, oM = 3, XO = 0, NSLOT = NSLOT_S;
  static constexpr int elem(int, int, int n) { return (n <= 4) ? 3 + n : ELEM_NONE; }
  __device__ static __forceinline__ void weights(const KParams& kp, const PairGeom<D>& g, double (&aw)[NJ]) {
    const double q = g.q;
    const double t = 2.0 - q;
    const double inner = fma(q * q, fma(kp.w_a, q, kp.w_b), kp.sigma_d);
    const double outer = ((kp.w_c * t) * t) * t;
    const double w = g.inner() ? inner : outer;
    aw[0] = g.hit ? w : 0.0;                       /* a miss: weight exactly 0 */
  }
  /* s: [NT][NJ][8] sums of this home */
  __device__ static void finish(const double* s, uint32_t cnt, const Sorted& so, int64_t i) {
    so.sigma_star[i] = s[0];
    so.s_star[i] = s[1];
    so.rho_star[0][i] = s[2];
    so.rho_star[1][i] = s[3];
    so.rho_star[2][i] = s[4];
    so.nnb[i] = cnt - 1u;     /* the home particle itself always passes (r2 = 0) */
  }
};

/* ------------------------------------------------------------------------------------------ a6 operator ---- */
/* Quantities of the gradient pass, numbered as "elements": m, then m times each of P, u[D], v[D], B[D*D], K[3*D],
   alpha[3] (written by the thermo kernel). */
struct GLayout { int M, P, U, V, B, K, AL, N; };
__host__ __device__ constexpr GLayout make_glayout(int D, bool visc, bool diff) {
  GLayout g{};
  g.M = 0; g.P = 1; g.U = 2; g.V = 2 + D; g.B = 2 + 2 * D;
  g.K = g.B + (visc ? D * D : 0);
  g.AL = g.K + (diff ? 3 * D : 0);
  g.N = g.AL + (diff ? 3 : 0);
  return g;
}
/* Column tiles (weight j = component of grad W):
     tile 0:  m | m P | m u_1..u_D | m alpha_B, alpha_S, alpha_Q (DIFF)       -> G_j, FP_j, DU_jk, DA_qj
              ( ideal fluid: | m v_j instead, so that one tile is enough )
     tile 1:  m v_j | m B_j1..B_jD (VISC) | m K_Bj, K_Sj, K_Qj (DIFF)          -> div v, FB_k, FK_q (summed over j at the end)
   grad_elem = element in column n of tile T for weight j. */
__host__ __device__ constexpr int grad_elem(int D, bool visc, bool diff, int T, int j, int n) {
  const GLayout L = make_glayout(D, visc, diff);
  const int NT = (visc || diff) ? 2 : 1;
  const int cDU = 2, cDA = 2 + D, cFB = 1, cFK = 1 + (visc ? D : 0);
  if (T == 0) {
    if (n == 0) return L.M;
    if (n == 1) return L.P;
    if (n < cDU + D) return L.U + (n - cDU);
    if (diff) return (n < cDA + 3) ? L.AL + (n - cDA) : ELEM_NONE;
    if (NT == 1 && n == 2 + D) return L.V + j;
    return ELEM_NONE;
  }
  if (n == 0) return L.V + j;
  if (visc && n >= cFB && n < cFB + D) return L.B + j * D + (n - cFB);
  if (diff && n >= cFK && n < cFK + 3) return L.K + (n - cFK) * D + j;
  return ELEM_NONE;
}
/* Record (32 doubles = 256 bytes): 8 blocks of 4 doubles, block n = the operands of MMA column n ("gid-major": the 4
   operands of lane (gid, tig) are 32 contiguous bytes, two 16-byte loads from one address): slot 0 = column n of tile 0,
   slots 1..3 = column n of tile 1 for j = 0, 1, 2 (viscous / diffusive), or slots 0..2 = column n of the single tile for
   j = 0, 1, 2 (ideal fluid: only its v_j column depends on j).  Slots 1..3 of block 7 are free in every variant (tile 1
   has at most 7 columns, the single tile of the ideal fluid at most 6) and hold the position x, y, z: the MMA column they
   feed is never read. */
constexpr int GREC_D = 32, GREC_B0 = 0, GREC_X = 29;
__host__ __device__ constexpr int grad_slot_elem(int D, bool visc, bool diff, int n, int s) {
  const bool two = visc || diff;
  const int T = two ? (s == 0 ? 0 : 1) : 0;
  const int j = two ? (s == 0 ? 0 : s - 1) : s;
  if (j >= D) return ELEM_NONE;
  return grad_elem(D, visc, diff, T, j, n);
}
/* position (double index in the record) of element e: its first appearance in the blocks */
__host__ __device__ constexpr int grad_pos(int D, bool visc, bool diff, int e) {
  for (int n = 0; n < 8; ++n)
    for (int s = 0; s < 4; ++s)
      if (grad_slot_elem(D, visc, diff, n, s) == e) return GREC_B0 + 4 * n + s;
  return -1;
}
/* 32-byte global store / load (sm_100: STG.256 / LDG.256); the address is 32-byte aligned */
__device__ __forceinline__ void st_global_v4(double* p, double a, double b, double c, double d) {
  asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(p), "d"(a), "d"(b), "d"(c), "d"(d) : "memory");
}
__device__ __forceinline__ void ldg_nc_v4(const double* p, double& a, double& b, double& c, double& d) {
  asm volatile("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(a), "=d"(b), "=d"(c), "=d"(d) : "l"(p));
}
#ifndef CCAKE_V4
#define CCAKE_V4 1
#endif
/* thermo kernel: scatter the elements el[0 .. L.N) of one particle into its record; pos: the position, which sits in the
   free slots 1..3 of block 7 */
template <int D, bool VISC, bool DIFF>
__device__ __forceinline__ void write_grad_record(double* __restrict__ rg, const double* el, const double (&pos)[3]) {
#pragma unroll
  for (int n = 0; n < 8; ++n) {
    double v[4];
#pragma unroll
    for (int s = 0; s < 4; ++s) {
      const int e = grad_slot_elem(D, VISC, DIFF, n, s);
      v[s] = (e >= 0) ? el[e] : 0.0;
      if (4 * n + s >= GREC_X) v[s] = pos[4 * n + s - GREC_X];
    }
#if CCAKE_V4
    st_global_v4(rg + GREC_B0 + 4 * n, v[0], v[1], v[2], v[3]);
#else
    reinterpret_cast<double2*>(rg + GREC_B0 + 4 * n)[0] = make_double2(v[0], v[1]);
    reinterpret_cast<double2*>(rg + GREC_B0 + 4 * n)[1] = make_double2(v[2], v[3]);
#endif
  }
}

template <int D_, bool VISC, bool DIFF>
struct GradOp {
  static constexpr int D = D_;
  static constexpr bool HASH = false, COUNT = false, GIDMAJOR = true, CARRY = CCAKE_PM_CARRY != 0;
  static constexpr int eM = make_glayout(D_, VISC, DIFF).M, eP = make_glayout(D_, VISC, DIFF).P, eU = make_glayout(D_, VISC, DIFF).U,
                       eV = make_glayout(D_, VISC, DIFF).V, eB = make_glayout(D_, VISC, DIFF).B, eK = make_glayout(D_, VISC, DIFF).K,
                       eAL = make_glayout(D_, VISC, DIFF).AL;
  static constexpr int NREC = GREC_D, XO = GREC_X, NSLOT = NSLOT_G;
  static constexpr int NJ = D, NT = (VISC || DIFF) ? 2 : 1;
  static constexpr int elem(int, int, int) { return ELEM_NONE; }       /* not used: the operands are found by position */
  /* column positions */
  static constexpr int cG = 0, cFP = 1, cDU = 2, cDA = 2 + D;
  static constexpr int tDV = NT - 1, cDV = (NT == 2) ? 0 : 2 + D, cFB = 1, cFK = 1 + (VISC ? D : 0);
  static constexpr int pos(int e) { return grad_pos(D_, VISC, DIFF, e); }
  /* the 4 operands of a lane -> B operand of tile T, weight j */
  __device__ static __forceinline__ void pick(const double2 b01, const double2 b23, double (&bop)[NT][NJ]) {
    const double b[4] = {b01.x, b01.y, b23.x, b23.y};
    if (NT == 2) {
#pragma unroll
      for (int j = 0; j < NJ; ++j) { bop[0][j] = b[0]; bop[NT - 1][j] = b[1 + j]; }
    } else {
#pragma unroll
      for (int j = 0; j < NJ; ++j) bop[0][j] = b[j];
    }
  }
  __device__ static __forceinline__ void weights(const KParams& kp, const PairGeom<D>& g, double (&aw)[NJ]) {
    /* Eq. 79: grad_i W = (sigma_D / h) f(q) dr_i / r,  f = -3q + 9/4 q^2 (q <= 1), -3/4 (2 - q)^2 (q <= 2) */
    const double t = 2.0 - g.q;
    const double fin = fma(kp.g_a, g.q, kp.g_b);                   /* f / r for q <= 1: no 1/r needed */
    const double fout = (t * t) * (kp.g_c * g.rinv);
    const double f = g.inner() ? fin : fout;
    const double fac = g.hit ? f : 0.0;                            /* a miss: weight exactly 0 */
#pragma unroll
    for (int k = 0; k < D; ++k) aw[k] = fac * g.dr[k];
  }
  /* combine with the home particle's own values: sum_b (A_a + A_b) dW = A_a G + sum_b A_b dW, etc.  The record
     holds m_a A_a. */
  __device__ static void finish(const double* s, uint32_t, const Sorted& so, int64_t i) {
    auto S = [&](int T, int j, int c) { return s[(T * NJ + j) * 8 + c]; };
    const double* __restrict__ ra = so.rec_g + i * NREC;
    const double inv = 1.0 / so.sigma_star[i];
    const double im = 1.0 / ra[pos(eM)];
    const double Pa = ra[pos(eP)] * im;
    double G[3] = {0.0, 0.0, 0.0};
    for (int k = 0; k < D; ++k) G[k] = S(0, k, cG);
    double dv = 0.0;
    for (int j = 0; j < D; ++j) dv += S(tDV, j, cDV);
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      double fp = 0.0, fb = 0.0;
      if (k < D) {
        fp = fma(Pa, G[k], S(0, k, cFP));
        if (VISC) {
          for (int j = 0; j < D; ++j) fb += S(1, j, cFB + k);
#pragma unroll
          for (int j = 0; j < D; ++j) fb = fma(ra[pos(VISC ? eB + j * D + (k < D ? k : 0) : 0)] * im, G[j], fb);
        }
        dv = fma(-(ra[pos(eV + (k < D ? k : 0))] * im), G[k], dv);
      }
      so.FP[k][i] = fp;
      so.FB[k][i] = fb;
    }
#pragma unroll
    for (int j = 0; j < 3; ++j)
#pragma unroll
      for (int k = 0; k < 3; ++k)
        so.DU[j * 3 + k][i] = (j < D && k < D) ? fma(-(ra[pos(eU + (k < D ? k : 0))] * im), G[j], S(0, j, cDU + k)) * inv : 0.0;
#pragma unroll
    for (int qq = 0; qq < 3; ++qq) {
      double fk = 0.0;
      if (DIFF) {
        for (int j = 0; j < D; ++j) fk += S(1, j, cFK + qq);
#pragma unroll
        for (int j = 0; j < D; ++j) fk = fma(ra[pos(DIFF ? eK + qq * D + j : 0)] * im, G[j], fk);
      }
      so.FK[qq][i] = fk;
#pragma unroll
      for (int j = 0; j < 3; ++j)
        so.DA[qq * 3 + j][i] = (DIFF && j < D) ? fma(-(ra[pos(DIFF ? eAL + qq : 0)] * im), G[j], S(0, j, cDA + qq)) * inv : 0.0;
    }
    so.divv[i] = dv * inv;
  }
};

/* ------------------------------------------------------------------------------ freeze-out operator ---- */
/* NEXT-2, §5.10 Eq. 147 (:1476): spatial gradient of the energy density by the n = +1 SPH
   derivative, d_i eps_a = (1/sigma*_a) sum_b m_b (eps_b - eps_a) d_i W_ab.  record: x[3], m, m eps, 0, 0, 0.
   Runs only when a freeze-out field is read (not on the step path). */
template <int D_>
struct EpsGradOp {
  static constexpr int D = D_;
  static constexpr bool HASH = false, COUNT = false, GIDMAJOR = false, CARRY = CCAKE_PM_CARRY != 0;
  static constexpr int NREC = 8, NJ = D, NT = 1, oM = 3, XO = 0, NSLOT = NSLOT_G;
  static constexpr int elem(int, int, int n) { return (n <= 1) ? 3 + n : ELEM_NONE; }
  __device__ static __forceinline__ void weights(const KParams& kp, const PairGeom<D>& g, double (&aw)[NJ]) {
    const double t = 2.0 - g.q;
    const double fin = fma(kp.g_a, g.q, kp.g_b);
    const double fout = (t * t) * (kp.g_c * g.rinv);
    const double f = g.inner() ? fin : fout;
    const double fac = g.hit ? f : 0.0;
#pragma unroll
    for (int k = 0; k < D; ++k) aw[k] = fac * g.dr[k];
  }
  __device__ static void finish(const double* s, uint32_t, const Sorted& so, int64_t i) {
    const double inv = 1.0 / so.sigma_star[i], ea = so.e[i];
    for (int k = 0; k < 3; ++k) so.fo_de[k][i] = (k < D) ? fma(-ea, s[k * 8 + 0], s[k * 8 + 1]) * inv : 0.0;
  }
};

/* ------------------------------------------------------------------------------------ shared memory ---- */
/* Tile: unit c (16 bytes = 2 doubles) of staged candidate k sits at unit index c * CSTRIDE + k with CSTRIDE = 1 mod 8
   (TILE_B + 1, plus the carry columns of the passes that have them), so its 16-byte bank group is (c + k) mod 8: the staging writes (consecutive c, same k) are
   conflict-free and the 8-byte operand reads of a quad (8 columns x 4 candidates) spread over the bank groups. */
template <class Op> struct PairCfg {
  static constexpr int NR = Op::NREC;
  static constexpr int NU = NR / 2;
  static constexpr int NSLOT = Op::NSLOT, TILE_B = NSLOT * HALF_B;
  static constexpr int NCARRY = Op::CARRY ? 3 * NGRP : 0;   /* carry columns behind the ring: 3 per group (a multiple of 8) */
  static constexpr int CARRY0 = TILE_B + 1;                 /* first carry column */
  static constexpr int CSTRIDE = TILE_B + 1 + NCARRY;
  static constexpr int FSTRIDE = HALF_B + 4;                /* FIFO entries per group: a tile and up to 3 carried candidates */
  static constexpr int NSUM = 8 * Op::NT * Op::NJ;          /* sums per home particle */
  static constexpr int SSTRIDE = NSUM + 2;                  /* scratch row of a home in the epilogue (even, skewed) */
  static constexpr size_t B_PAY = sizeof(double2) * NU * CSTRIDE;
  static constexpr size_t B_PAYX = sizeof(float4) * TILE_B;
  static constexpr size_t B_LIST = sizeof(uint32_t) * (LCAP + LB * PT);
  static constexpr size_t B_FIFO = sizeof(uint16_t) * NGRP * FSTRIDE;  /* tile entries waiting per group */
  static constexpr size_t B_MASK = sizeof(uint4) * NSLOT * NGRP;
  static constexpr size_t B_RING = B_PAY + B_PAYX + B_LIST + B_FIFO + B_MASK;
  static constexpr size_t B_SCRATCH = sizeof(double) * BH * SSTRIDE;
  static constexpr size_t SMEM = (B_RING > B_SCRATCH) ? B_RING : B_SCRATCH;
};

/* ------------------------------------------------------------------------------------ candidate lists ---- */
/* Once per substep, for every pair block (BH consecutive home particles): the sorted slots of all particles of the
   cell rows overlapping the block's bounding box +- 2h that pass the FP32 test against that box (conservative
   margin, Grid::cutm2), in ascending (row, slot) order — kept with ballots and a block scan, no atomics, so the
   list and everything summed along it is reproducible.  Both pair passes of the substep read it.  A block whose
   list does not fit cand_cap entries is marked 0xffffffff and lists its candidates inside the pass instead. */
template <int D>
__global__ void __launch_bounds__(BH)
cand_list_kernel(int64_t n, const Grid* __restrict__ grid, Sorted so) {
  constexpr int NW = BH / 32, LBK = CCAKE_CL_LBK;
  __shared__ float s_lo[NW][3], s_hi[NW][3];
  __shared__ int wcnt[LBK * NW];
  __shared__ uint32_t rb0[MAXROW], rcum[MAXROW + 1];
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  const float4* __restrict__ xf = so.xf;
  const int64_t i = (int64_t)blockIdx.x * BH + tid;
  const float4 fa = xf[(i < n) ? i : n - 1];
  float blo[3], bhi[3];
  {
    float lo[3] = {fa.x, fa.y, (D == 3) ? fa.z : 0.f}, hi[3] = {fa.x, fa.y, (D == 3) ? fa.z : 0.f};
#pragma unroll
    for (int k = 0; k < 3; ++k) { lo[k] = warp_minf(lo[k]); hi[k] = warp_maxf(hi[k]); }
    if (lane == 0)
      for (int k = 0; k < 3; ++k) { s_lo[w][k] = lo[k]; s_hi[w][k] = hi[k]; }
    __syncthreads();
    for (int k = 0; k < 3; ++k) {
      blo[k] = s_lo[0][k]; bhi[k] = s_hi[0][k];
      for (int j = 1; j < NW; ++j) { blo[k] = fminf(blo[k], s_lo[j][k]); bhi[k] = fmaxf(bhi[k], s_hi[j][k]); }
    }
  }
  const Grid g = *grid;
  const float cutm2 = g.cutm2;
  int c0[3] = {0, 0, 0}, c1[3] = {0, 0, 0};
#pragma unroll
  for (int k = 0; k < D; ++k) {
    const double lo = ((double)blo[k] - g.cutm) * g.inv_edge, hi = ((double)bhi[k] + g.cutm) * g.inv_edge;
    c0[k] = (lo > 0.0) ? min((int)lo, g.nc[k] - 1) : 0;
    c1[k] = (hi > 0.0) ? min((int)hi, g.nc[k] - 1) : 0;
  }
  uint32_t* __restrict__ out = so.cand_list + (size_t)blockIdx.x * so.cand_cap;
  const uint32_t cap = (uint32_t)so.cand_cap;
  uint32_t nrel = 0;
  const int ny = c1[1] - c0[1] + 1, nrows = ny * (c1[2] - c0[2] + 1);
#pragma unroll 1
  for (int r0 = 0; r0 < nrows; r0 += MAXROW) {
    const int nr = min(MAXROW, nrows - r0);
    __syncthreads();
    if (tid < nr) {
      const int rr = r0 + tid, cz = c0[2] + rr / ny, cy = c0[1] + rr % ny;
      int cfirst, clast;
      snake_range(g, snake_row(g, cy, cz), c0[0], c1[0], cfirst, clast);
      const uint32_t b0 = so.cell_start[cfirst], b1 = so.cell_start[clast + 1];
      rb0[tid] = b0;
      rcum[tid + 1] = b1 - b0;
    }
    __syncthreads();
    if (tid == 0) {
      rcum[0] = 0;
      for (int r = 0; r < nr; ++r) rcum[r + 1] += rcum[r];
    }
    __syncthreads();
    const uint32_t raw = rcum[nr];
    int rowh[LBK];                                   /* row of the thread's previous entry: f only grows, and a row holds
                                                        hundreds of entries, so the search is a step or two from there */
#pragma unroll
    for (int u = 0; u < LBK; ++u) rowh[u] = 0;
#pragma unroll 1
    for (uint32_t fb = 0; fb < raw; fb += LBK * BH) {
      bool r[LBK];
      uint32_t j[LBK], bal[LBK];
#pragma unroll
      for (int u = 0; u < LBK; ++u) {
        const uint32_t f = fb + (uint32_t)(u * BH + tid);
        r[u] = false;
        j[u] = 0;
        if (f < raw) {
          int row = rowh[u];                          /* the last row with rcum[row] <= f (rcum is monotone) */
          while (row + 1 < nr && rcum[row + 1] <= f) ++row;
          rowh[u] = row;
          j[u] = rb0[row] + (f - rcum[row]);
          r[u] = box_dist2<D>(xf[j[u]], blo, bhi) <= cutm2;
        }
      }
#pragma unroll
      for (int u = 0; u < LBK; ++u) {
        bal[u] = __ballot_sync(0xffffffffu, r[u]);
        if (lane == 0) wcnt[u * NW + w] = __popc(bal[u]);
      }
      __syncthreads();
      uint32_t tot = 0;
#pragma unroll
      for (int u = 0; u < LBK; ++u) {
        uint32_t off = nrel + tot;
#pragma unroll
        for (int q = 0; q < NW; ++q) { const uint32_t cq = (uint32_t)wcnt[u * NW + q]; off += (q < w) ? cq : 0u; tot += cq; }
        off += __popc(bal[u] & ((1u << lane) - 1u));
        if (r[u] && off < cap) out[off] = j[u];
      }
      nrel += tot;
      __syncthreads();
    }
  }
  if (tid == 0) so.cand_cnt[blockIdx.x] = (nrel <= cap) ? nrel : 0xffffffffu;
}

#ifdef CCAKE_PAIR_PROF
/* experiment builds only: [0] quads of all warps, [1] sum over blocks of (warps x max quads of a warp), per pass kind */
__device__ unsigned long long g_pair_prof[16];
#endif

__device__ __forceinline__ uint64_t pm_mix64(uint64_t z) {      /* splitmix64 finaliser (include/ccake.h) */
  z += 0x9E3779B97F4A7C15ULL;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
  return z ^ (z >> 31);
}

/* ------------------------------------------------------------------------------------------ the kernel ---- */
/* MC: 0 = the hit masks are computed and used here; 1 = also stored, refined to the exact union of the group's
   neighbour sets (smoothing pass); 2 = read back (later passes of the same substep: same positions, same sorted
   order, same block / tile / group numbering). */
template <class Op, int MC>
__global__ void __launch_bounds__(PT, PM_MINB)
pair_mma_kernel(int64_t n, KParams kp, const Grid* __restrict__ grid, Sorted so, const double* __restrict__ rec,
                const uint32_t* __restrict__ orig, unsigned long long* __restrict__ hash_out) {
  constexpr int D = Op::D;
  constexpr int NU = PairCfg<Op>::NU;
  constexpr int CSTRIDE = PairCfg<Op>::CSTRIDE;
  constexpr int NSLOT = PairCfg<Op>::NSLOT, TILE_B = PairCfg<Op>::TILE_B;
  constexpr int NW = PM_WARPS, GPW = PM_GPW, NJ = Op::NJ, NT = Op::NT;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double2* pay = reinterpret_cast<double2*>(smem_raw);                  /* [NU][CSTRIDE] staged records        */
  float4* payx = reinterpret_cast<float4*>(pay + NU * CSTRIDE);         /* [TILE_B] FP32 positions of the tile */
  uint32_t* list = reinterpret_cast<uint32_t*>(payx + TILE_B);          /* [LCAP + LB * PT] block candidate list */
  uint16_t* fifo = reinterpret_cast<uint16_t*>(list + LCAP + LB * PT);  /* [NGRP][FSTRIDE] byte offsets of the staged entries that passed, per group */
  uint4* mstage = reinterpret_cast<uint4*>(fifo + NGRP * PairCfg<Op>::FSTRIDE);       /* [NSLOT][NGRP] cached hit masks of the staged tiles (MC == 2) */
  __shared__ float s_lo[NW][3], s_hi[NW][3];
  __shared__ int wcnt[LB * NW];
  __shared__ uint32_t rb0[MAXROW], rcum[MAXROW + 1];
  __shared__ __align__(8) unsigned long long full_bar[NSLOT];      /* mbarrier: the copies of the slot's tile landed */
  __shared__ volatile int done_turn[NW];                           /* last turn (tile number) each warp finished */

  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  const int gid = lane >> 2, tig = lane & 3;        /* MMA fragment coordinates: home row / column, candidate */
  const uint32_t lt_mask = (1u << lane) - 1u;
  const uint32_t tig_bit = 1u << tig;
  const float4* __restrict__ xf = so.xf;

  /* the lane's home particle in each of the warp's groups (4 lanes share one); tail lanes shadow the last particle
     and write nothing */
  int64_t ih[GPW];
  double xa[GPW][3];
  float scx[GPW], scy[GPW], scz[GPW], shx[GPW], shy[GPW], shz[GPW];   /* FP32 box of the group: centre, half-extent */
  float blo[3], bhi[3];
  {
    float lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
#pragma unroll
    for (int g = 0; g < GPW; ++g) {
      ih[g] = (int64_t)blockIdx.x * BH + (w * GPW + g) * 8 + gid;
      const int64_t ic = (ih[g] < n) ? ih[g] : n - 1;
      xa[g][0] = xa[g][1] = xa[g][2] = 0.0;
#pragma unroll
      for (int k = 0; k < D; ++k) xa[g][k] = rec[ic * Op::NREC + Op::XO + k];
      const float4 fa = xf[ic];
      float glo[3] = {fa.x, fa.y, (D == 3) ? fa.z : 0.f}, ghi[3] = {fa.x, fa.y, (D == 3) ? fa.z : 0.f};
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        glo[k] = warp_minf(glo[k]); ghi[k] = warp_maxf(ghi[k]);
        lo[k] = fminf(lo[k], glo[k]); hi[k] = fmaxf(hi[k], ghi[k]);
      }
      /* centre / half-extent rounded so that [c - h, c + h] contains [lo, hi] */
      scx[g] = 0.5f * (glo[0] + ghi[0]); shx[g] = __fmul_ru(fmaxf(ghi[0] - scx[g], scx[g] - glo[0]), 1.000001f);
      scy[g] = 0.5f * (glo[1] + ghi[1]); shy[g] = __fmul_ru(fmaxf(ghi[1] - scy[g], scy[g] - glo[1]), 1.000001f);
      scz[g] = 0.5f * (glo[2] + ghi[2]); shz[g] = __fmul_ru(fmaxf(ghi[2] - scz[g], scz[g] - glo[2]), 1.000001f);
    }
    if (lane == 0)
      for (int k = 0; k < 3; ++k) { s_lo[w][k] = lo[k]; s_hi[w][k] = hi[k]; }
    __syncthreads();
    for (int k = 0; k < 3; ++k) {
      blo[k] = s_lo[0][k]; bhi[k] = s_hi[0][k];
      for (int j = 1; j < NW; ++j) { blo[k] = fminf(blo[k], s_lo[j][k]); bhi[k] = fmaxf(bhi[k], s_hi[j][k]); }
    }
  }
  const Grid g = *grid;
  const float cutm2 = g.cutm2;

  if (tid < NSLOT) {
    const uint32_t a = (uint32_t)__cvta_generic_to_shared(&full_bar[tid]);
    asm volatile("mbarrier.init.shared.b64 [%0], %1;" ::"r"(a), "r"(PT));
  }
  if (tid < NW) done_turn[tid] = -1;
  __syncthreads();

  /* byte offsets of this lane's B operands inside a staged record: column gid of tile T for weight j.  They live in
     a small table in shared memory and are read back in front of every quad loop: kept in registers across the
     culling and compaction code the compiler recomputed them per tile with a chain of ~60 selects */
  const uint32_t pay_s = (uint32_t)__cvta_generic_to_shared(pay);
  const uint32_t payx_s = (uint32_t)__cvta_generic_to_shared(payx);
  __shared__ uint32_t s_boff[NT * NJ][8];
  if (tid < 8) {
#pragma unroll
    for (int T = 0; T < NT; ++T)
#pragma unroll
      for (int j = 0; j < NJ; ++j) {
        int e = ELEM_NONE;
#pragma unroll
        for (int c = 0; c < 8; ++c) if (c == tid) e = Op::elem(T, j, c);
        if (e < 0) e = 0;                            /* unused column: any finite element; its sums are dropped */
        s_boff[T * NJ + j][tid] = (uint32_t)((e >> 1) * CSTRIDE) * 16u + (uint32_t)(e & 1) * 8u;
      }
  }
  __syncthreads();
  const uint32_t lane_goff = (uint32_t)((GREC_B0 / 2 + 2 * gid) * CSTRIDE) * 16u;   /* GIDMAJOR: byte offset of the lane's operands */
  uint32_t boff[NT][NJ];
  auto load_boff = [&]() {
    if constexpr (!Op::GIDMAJOR) {
#pragma unroll
      for (int T = 0; T < NT; ++T)
#pragma unroll
        for (int j = 0; j < NJ; ++j) boff[T][j] = *reinterpret_cast<volatile uint32_t*>(&s_boff[T * NJ + j][gid]);
    }
  };
  load_boff();

  double acc[GPW][NT][NJ][2];
#pragma unroll
  for (int gg = 0; gg < GPW; ++gg)
#pragma unroll
    for (int T = 0; T < NT; ++T)
#pragma unroll
      for (int j = 0; j < NJ; ++j) acc[gg][T][j][0] = acc[gg][T][j][1] = 0.0;
  uint32_t hits[GPW];
  unsigned long long hsum[GPW];
#pragma unroll
  for (int gg = 0; gg < GPW; ++gg) { hits[gg] = 0u; hsum[gg] = 0ull; }
  int nrel = 0;
#ifdef CCAKE_PAIR_PROF
  unsigned prof_quads = 0;
#endif

  /* one quad: lane (gid, tig) evaluates the pair (home gid of the group, candidate tig of the quad) and the warp
     accumulates 8 homes x 4 candidates x 8 columns per MMA.  koff: byte offset of the lane's candidate in the ring.  Returns
     (smoothing pass) the 4 bits "candidate t of the quad is within 2h of at least one home of the group". */
  auto quad = [&](const int gg, const uint32_t koff, const bool act) -> uint32_t {
    const double2* __restrict__ p = reinterpret_cast<const double2*>(reinterpret_cast<const unsigned char*>(pay) + koff);
    double xb, yb, zb;
    if constexpr (Op::GIDMAJOR) {                       /* x in the upper half of unit 14, (y, z) = unit 15 */
      xb = reinterpret_cast<const double*>(p + (GREC_X / 2) * CSTRIDE)[1];
      const double2 yz = p[(GREC_X / 2 + 1) * CSTRIDE];
      yb = yz.x; zb = (D == 3) ? yz.y : 0.0;
    } else {
      const double2 h0 = p[0];
      xb = h0.x; yb = h0.y;
      zb = (D == 3) ? reinterpret_cast<const double*>(p + CSTRIDE)[0] : 0.0;
    }
    PairGeom<D> pg;
    pg.set(kp, xa[gg], xb, yb, zb, act);
    double aw[NJ], bop[NT][NJ];
    Op::weights(kp, pg, aw);
    const unsigned char* rb = reinterpret_cast<const unsigned char*>(p);
    if constexpr (Op::GIDMAJOR) {
      const double2* pl = reinterpret_cast<const double2*>(rb + lane_goff);       /* units 2 + 2 gid and the next one */
      Op::pick(pl[0], pl[CSTRIDE], bop);
    } else {
#pragma unroll
      for (int T = 0; T < NT; ++T)
#pragma unroll
        for (int j = 0; j < NJ; ++j) bop[T][j] = *reinterpret_cast<const double*>(rb + boff[T][j]);
    }
    if (Op::COUNT) hits[gg] += pg.hit ? 1u : 0u;
    if (Op::HASH) {
      const uint32_t slot = __float_as_uint(payx[koff >> 4].w);  /* sorted slot of the candidate (pack_smoothing_kernel) */
      if (pg.hit && (int64_t)slot != ih[gg]) hsum[gg] += pm_mix64((uint64_t)orig[so.perm[slot]] + 1ULL);
    }
    uint32_t nib = 0u;
    if (MC == 1) nib = __reduce_or_sync(0xffffffffu, pg.hit ? tig_bit : 0u);
#pragma unroll
    for (int T = 0; T < NT; ++T)
#pragma unroll
      for (int j = 0; j < NJ; ++j) dmma_m8n8k4(acc[gg][T][j][0], acc[gg][T][j][1], aw[j], bop[T][j]);
    return nib;
  };

  const double2* __restrict__ rec2 = reinterpret_cast<const double2*>(rec);
  int tt = 0;                                       /* tiles consumed so far: tile number tt lives in slot tt % NSLOT */
  /* hit-mask cache: [block][tile][group] x 128 bit */
  const int mtiles = (MC != 0 && so.mask_cache != nullptr) ? so.mask_tiles : 0;
  uint4* __restrict__ mrow = reinterpret_cast<uint4*>(so.mask_cache) + (size_t)blockIdx.x * (size_t)max(mtiles, 1) * NGRP;
  /* the candidates come from the global list of this block (cand_list_kernel) or, if that is absent or did not
     fit, from the list in shared memory filled further below */
  const uint32_t gcnt = (so.cand_cap > 0) ? so.cand_cnt[blockIdx.x] : 0xffffffffu;
  const bool use_glist = gcnt != 0xffffffffu;
  const uint32_t* __restrict__ lsrc = use_glist ? so.cand_list + (size_t)blockIdx.x * so.cand_cap : list;

  /* list entry of the tile-t record this lane owns (lane r < RPW of warp w owns entry w * RPW + r), or none: loaded
     before it is needed, so the L2 latency of the list is off the critical path */
  auto load_j = [&](const int cnt, const int ntile, const int t) {
    uint32_t j = 0xffffffffu;
    if (lane < RPW && t < ntile) {
      const int e = (w * RPW + lane) * ntile + t;
      if (e < cnt) j = lsrc[e];
    }
    return j;
  };
  const uint32_t mstage_s = (uint32_t)__cvta_generic_to_shared(mstage);
  auto issue = [&](const uint32_t j, const int slot, const bool need_x, const int u) {
    /* warp w copies entries [w * RPW, (w + 1) * RPW) of the tile: FP32 position (a 16-byte copy by the owning lane) and
       the records unit by unit, consecutive lanes taking consecutive units (coalesced rows) */
    const int sb = slot * HALF_B;
    if (MC == 2 && !need_x && lane < GPW)           /* the cached hit masks of the warp's groups travel with the tile */
      asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(mstage_s + (uint32_t)(slot * NGRP + w * GPW + lane) * 16u),
                   "l"(mrow + (size_t)u * NGRP + (w * GPW + lane)));
    if (need_x && j != 0xffffffffu)                 /* padding entries keep stale data; the masks leave them out */
      asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(payx_s + (uint32_t)(sb + w * RPW + lane) * 16u), "l"(xf + j));
#pragma unroll
    for (int i = 0; i < (RPW * NU + 31) / 32; ++i) {
      const int idx = i * 32 + lane;                  /* unit index within the warp's RPW records */
      const int r = idx / NU, c = idx - r * NU;
      const uint32_t jr = __shfl_sync(0xffffffffu, j, r & 31);
      if (idx < RPW * NU && jr != 0xffffffffu)
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(pay_s + (uint32_t)(c * CSTRIDE + sb + w * RPW + r) * 16u),
                     "l"(rec2 + (int64_t)jr * NU + c));
    }
    /* the slot's mbarrier gets this thread's arrival when all its copies above have landed */
    asm volatile("cp.async.mbarrier.arrive.noinc.shared.b64 [%0];" ::"r"((uint32_t)__cvta_generic_to_shared(&full_bar[slot])));
  };
  /* every warp has finished turn `turn` (tile numbers; -1 before the first) */
  auto all_done = [&](const int turn) {
    int d = done_turn[lane % NW];
    d = __reduce_min_sync(0xffffffffu, d);
    return d >= turn;
  };

  /* consume list[0..cnt): tiles of up to HALF_B candidates taken with stride ntile through the list, so that every
     tile samples the whole neighbourhood of the block and all groups find about the same number of hits in it.
     The tiles live in a ring of NSLOT slots.  Every warp copies its share of every tile (cp.async; an mbarrier per
     slot collects the arrivals), as far ahead as the ring allows: tile u goes into the slot of tile u - NSLOT, which
     must have been consumed by every warp (done_turn).  A warp never waits for the others except for data: there is
     no block barrier per tile, and a warp may run up to NSLOT - 1 tiles ahead of the slowest one. */
  auto flush = [&](const int cnt) {
    const int ntile = (cnt + HALF_B - 1) / HALF_B;
    const int tt0 = tt;
    /* entries of tile t: tq, one more if t < trm.  The smoothing pass keeps (tq, trm) instead of dividing per tile (8.05 ->
       8.00 ms on C4); in the gradient pass the two live registers cost more than the division (12.17 -> 12.21 ms) */
    constexpr bool NODIV = (MC == 1);
    const int tq = NODIV ? cnt / max(ntile, 1) : 0, trm = NODIV ? cnt - tq * ntile : 0;
    /* CARRY: the tl & 3 candidates of a tile that do not fill a quad are not evaluated as a partial quad (a whole quad's cost
       for 2.5 candidates on average, once per tile and group); their records are copied into the group's 3 carry columns
       behind the ring and lead the FIFO of the next tile.  Only the last tile of a flush ends with a partial quad.  (Not in
       the smoothing pass: its union masks are per tile.) */
    constexpr bool CARRY = Op::CARRY && MC == 2;
    int ncarry[GPW];
#pragma unroll
    for (int gg = 0; gg < GPW; ++gg) ncarry[gg] = 0;
    int ni = 0;                                                   /* next tile of this flush the warp has to issue */
    uint32_t jn = load_j(cnt, ntile, 0);
    auto try_issue = [&](const int upto, const bool block) {
      while (ni <= upto && ni < ntile) {
        const int u = tt0 + ni;
        if (!all_done(u - NSLOT)) {
          if (!block) break;
          do { __nanosleep(1000); } while (!all_done(u - NSLOT));
        }
        issue(jn, u % NSLOT, MC != 2 || u >= mtiles, u);
        ++ni;
        jn = load_j(cnt, ntile, ni);
      }
    };
#pragma unroll 1
    for (int t = 0; t < ntile; ++t, ++tt) {
      const int tcnt = NODIV ? tq + ((t < trm) ? 1 : 0)
                             : (cnt - t + ntile - 1) / ntile;     /* entries e = m * ntile + t < cnt, m < tcnt */
      const int sb = (tt % NSLOT) * HALF_B;                       /* first slot of this tile */
      try_issue(t + NSLOT - 1, false);
      try_issue(t, true);
      {                                                           /* wait for the copies of tile tt */
        const uint32_t a = (uint32_t)__cvta_generic_to_shared(&full_bar[tt % NSLOT]);
        const uint32_t parity = (uint32_t)((tt / NSLOT) & 1);
        uint32_t ok = 0;
        while (!ok)                                               /* the hint lets the hardware park the warp */
          asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared.b64 p, [%1], %2, %3; selp.u32 %0, 1, 0, p; }"
                       : "=r"(ok) : "r"(a), "r"(parity), "r"(20000u) : "memory");
      }
      const bool cached = (MC != 0) && tt < mtiles;
#pragma unroll
      for (int gg = 0; gg < GPW; ++gg) {
        uint16_t* ff = fifo + (w * GPW + gg) * PairCfg<Op>::FSTRIDE;
        /* survivors of the tile for this group: the cached exact-union mask, or the FP32 test against the group box */
        uint32_t bal[NR32];
        if (MC == 2 && cached) {
          const uint4 mw = mstage[(tt % NSLOT) * NGRP + (w * GPW + gg)];
          bal[0] = mw.x;
          if (NR32 > 1) bal[1 % NR32] = mw.y;
          if (NR32 > 2) bal[2 % NR32] = mw.z;
          if (NR32 > 3) bal[3 % NR32] = mw.w;
        } else {
#pragma unroll
          for (int r = 0; r < NR32; ++r) {
            const int k = r * 32 + lane;
            const float4 fb = payx[sb + k];
            const float dx = fmaxf(fabsf(fb.x - scx[gg]) - shx[gg], 0.f), dy = fmaxf(fabsf(fb.y - scy[gg]) - shy[gg], 0.f);
            float d2 = dx * dx + dy * dy;
            if (D == 3) { const float dz = fmaxf(fabsf(fb.z - scz[gg]) - shz[gg], 0.f); d2 += dz * dz; }
            bal[r] = __ballot_sync(0xffffffffu, k < tcnt && d2 <= cutm2);   /* entries beyond tcnt are padding */
          }
        }
        /* compaction, ascending: entry k of the tile goes to position pos[r] */
        int pos[NR32], tl = CARRY ? ncarry[gg] : 0;               /* the carried candidates are ff[0 .. ncarry) already */
#pragma unroll
        for (int r = 0; r < NR32; ++r) {
          pos[r] = tl + __popc(bal[r] & lt_mask);
          if ((bal[r] >> lane) & 1u) ff[pos[r]] = (uint16_t)((sb + r * 32 + lane) * 16);
          tl += __popc(bal[r]);
        }
        __syncwarp();
        /* full quads, then one partial quad (idle lanes re-read its first candidate with weight 0) */
        load_boff();
        uint32_t nibs = 0u;                                       /* lane q: the 4 union bits of quad q */
        const int nfull = tl >> 2;
        const uint16_t* fq = ff + tig;
        if (MC == 1) {
#pragma unroll 1
          for (int q = 0; q < nfull; ++q) {
            const uint32_t nib = quad(gg, fq[4 * q], true);
            nibs = (lane == q) ? nib : nibs;
          }
        } else {
          const uint16_t* fend = fq + 4 * nfull;
#pragma unroll 1
          for (const uint16_t* fp = fq; fp != fend; fp += 4) quad(gg, *fp, true);
        }
        if (CARRY && t + 1 < ntile) {
          const int rem = tl & 3;
          if (rem) {
            /* left-over i (FIFO entry 4 nfull + i) -> carry column i of this group, NU units each.  With nfull == 0 the
               first ncarry entries are carried ones and sit in their columns already; all others come from the ring. */
            constexpr int NCP = (3 * NU + 31) / 32;
            const uint32_t cbase = (uint32_t)(PairCfg<Op>::CARRY0 + (w * GPW + gg) * 3) * 16u;
            const int ci0 = (nfull == 0) ? ncarry[gg] : 0;
#pragma unroll
            for (int x = 0; x < NCP; ++x) {
              const int idx = x * 32 + lane, ci = idx / NU, cu = idx - ci * NU;
              if (ci >= ci0 && ci < rem) {
                unsigned char* col = reinterpret_cast<unsigned char*>(pay) + (size_t)cu * CSTRIDE * 16;
                *reinterpret_cast<double2*>(col + cbase + (uint32_t)ci * 16u) = *reinterpret_cast<const double2*>(col + ff[4 * nfull + ci]);
              }
            }
            __syncwarp();
            if (lane < rem) ff[lane] = (uint16_t)(cbase + (uint32_t)lane * 16u);
          }
          ncarry[gg] = rem;
        } else if (tl & 3) {
          const bool act = 4 * nfull + tig < tl;
          const uint32_t nib = quad(gg, ff[act ? 4 * nfull + tig : 4 * nfull], act);
          if (MC == 1) nibs = (lane == nfull) ? nib : nibs;
        }
        if (MC == 1 && cached) {
          /* exact union of the group's neighbour sets for this tile: the box mask minus the candidates that hit no home */
          uint32_t wd[4] = {0u, 0u, 0u, 0u};
#pragma unroll
          for (int r = 0; r < NR32; ++r) {
            const uint32_t nb = __shfl_sync(0xffffffffu, nibs, pos[r] >> 2);
            wd[r] = __ballot_sync(0xffffffffu, ((bal[r] >> lane) & 1u) && ((nb >> (pos[r] & 3)) & 1u));
          }
          if (lane == 0) mrow[(size_t)tt * NGRP + (w * GPW + gg)] = make_uint4(wd[0], wd[1], wd[2], wd[3]);
        }
        __syncwarp();
      }
      if (lane == 0) { __threadfence_block(); done_turn[w] = tt; }
    }
    __syncthreads();                                              /* the list may be refilled */
  };

  if (use_glist) {
    flush((int)gcnt);                               /* one flush: every tile samples the whole neighbourhood */
  } else {
    /* Candidate listing inside the pass.  The rows of cells that overlap the block box (batches of up to MAXROW rows)
       are treated as one flat index space f = 0 .. raw-1 (row r owns [rcum[r], rcum[r+1]), sorted slot j = rb0[r] +
       f - rcum[r]).  The list holds LCAP entries, fewer than a block's neighbourhood; so that every flush is still a
       uniform sample of the WHOLE neighbourhood, the space is swept NP times, sweep p taking f = p, p + NP, ...
       Every step tests LB * PT candidates against the block box and keeps them in order with ballots. */
    int c0[3] = {0, 0, 0}, c1[3] = {0, 0, 0};
#pragma unroll
    for (int k = 0; k < D; ++k) {
      const double lo = ((double)blo[k] - g.cutm) * g.inv_edge, hi = ((double)bhi[k] + g.cutm) * g.inv_edge;
      c0[k] = (lo > 0.0) ? min((int)lo, g.nc[k] - 1) : 0;
      c1[k] = (hi > 0.0) ? min((int)hi, g.nc[k] - 1) : 0;
    }
    const int ny = c1[1] - c0[1] + 1, nrows = ny * (c1[2] - c0[2] + 1);
#pragma unroll 1
    for (int r0 = 0; r0 < nrows; r0 += MAXROW) {
      const int nr = min(MAXROW, nrows - r0);
      __syncthreads();
      if (tid < nr) {
        const int rr = r0 + tid, cz = c0[2] + rr / ny, cy = c0[1] + rr % ny;
        int cfirst, clast;
        snake_range(g, snake_row(g, cy, cz), c0[0], c1[0], cfirst, clast);
        const uint32_t b0 = so.cell_start[cfirst], b1 = so.cell_start[clast + 1];
        rb0[tid] = b0;
        rcum[tid + 1] = b1 - b0;
      }
      __syncthreads();
      if (tid == 0) {
        rcum[0] = 0;
        for (int r = 0; r < nr; ++r) rcum[r + 1] += rcum[r];
      }
      __syncthreads();
      const uint32_t raw = rcum[nr];
      const uint32_t NP = max(1u, (raw + (LCAP * 3) / 4 - 1) / ((LCAP * 3) / 4));
#pragma unroll 1
      for (uint32_t pz = 0; pz < NP; ++pz) {
#pragma unroll 1
        for (uint32_t fb = pz; fb < raw; fb += LB * PT * NP) {
          bool r[LB];
          uint32_t j[LB], bal[LB];
#pragma unroll
          for (int u = 0; u < LB; ++u) {
            const uint32_t f = fb + (uint32_t)(u * PT + tid) * NP;
            r[u] = false;
            j[u] = 0;
            if (f < raw) {
              int row = 0;
#pragma unroll
              for (int st = MAXROW / 2; st > 0; st >>= 1) {                   /* rcum is monotone: binary search */
                const int rq = row + st;
                if (rq < nr && rcum[rq] <= f) row = rq;
              }
              j[u] = rb0[row] + (f - rcum[row]);
              r[u] = box_dist2<D>(xf[j[u]], blo, bhi) <= cutm2;
            }
          }
#pragma unroll
          for (int u = 0; u < LB; ++u) {
            bal[u] = __ballot_sync(0xffffffffu, r[u]);
            if (lane == 0) wcnt[u * NW + w] = __popc(bal[u]);
          }
          __syncthreads();
          int tot = 0;
#pragma unroll
          for (int u = 0; u < LB; ++u) {
            int off = nrel + tot;
#pragma unroll
            for (int q = 0; q < NW; ++q) { const int cq = wcnt[u * NW + q]; off += (q < w) ? cq : 0; tot += cq; }
            if (r[u]) list[off + __popc(bal[u] & lt_mask)] = j[u];
          }
          nrel += tot;
          __syncthreads();
          if (nrel >= LCAP) {
            flush(LCAP);
            const int rest = nrel - LCAP;           /* < LB * PT */
            uint32_t keep = 0;
            if (tid < rest) keep = list[LCAP + tid];
            __syncthreads();
            if (tid < rest) list[tid] = keep;
            nrel = rest;
            __syncthreads();
          }
        }
        if (nrel > 0) { flush(nrel); nrel = 0; }
      }
    }
  }

#ifdef CCAKE_PAIR_PROF
  {
    __shared__ unsigned int p_max, p_sum;
    if (tid == 0) { p_max = 0; p_sum = 0; }
    __syncthreads();
    if (lane == 0) { atomicMax(&p_max, prof_quads); atomicAdd(&p_sum, prof_quads); }
    __syncthreads();
    if (tid == 0) {
      const int base = (MC == 1) ? 0 : 4;
      atomicAdd(&g_pair_prof[base + 0], (unsigned long long)p_sum);
      atomicAdd(&g_pair_prof[base + 1], (unsigned long long)p_max * NW);
      atomicAdd(&g_pair_prof[base + 2], 1ull);
    }
  }
#endif
  /* epilogue: the sums of every home go through shared memory (the ring is no longer needed) so that one thread
     finishes one home particle and the stores are coalesced */
  __syncthreads();
  double* scratch = reinterpret_cast<double*>(smem_raw);
  constexpr int SS = PairCfg<Op>::SSTRIDE;
#pragma unroll
  for (int gg = 0; gg < GPW; ++gg) {
    double* row = scratch + ((w * GPW + gg) * 8 + gid) * SS;
#pragma unroll
    for (int T = 0; T < NT; ++T)
#pragma unroll
      for (int j = 0; j < NJ; ++j)
        *reinterpret_cast<double2*>(row + (T * NJ + j) * 8 + 2 * tig) = make_double2(acc[gg][T][j][0], acc[gg][T][j][1]);
    if (Op::COUNT || Op::HASH) {
      uint32_t c = hits[gg];
      c += __shfl_xor_sync(0xffffffffu, c, 1);
      c += __shfl_xor_sync(0xffffffffu, c, 2);
      unsigned long long hs = hsum[gg];
      hs += __shfl_xor_sync(0xffffffffu, hs, 1);
      hs += __shfl_xor_sync(0xffffffffu, hs, 2);
      if (tig == 0) {
        row[PairCfg<Op>::NSUM] = __longlong_as_double((long long)c);
        if (Op::HASH && ih[gg] < n) hash_out[orig[so.perm[ih[gg]]]] = hs;
      }
    }
  }
  __syncthreads();
  if (tid < BH) {
    const int64_t i = (int64_t)blockIdx.x * BH + tid;
    if (i < n) {
      const double* row = scratch + tid * SS;
      const uint32_t c = (Op::COUNT) ? (uint32_t)__double_as_longlong(row[PairCfg<Op>::NSUM]) : 0u;
      Op::finish(row, c, so, i);
    }
  }
}

template <class Op, int MC>
int launch_pair(int64_t N, const KParams& kp, const Grid* grid, const Sorted& so, const double* rec, cudaStream_t st,
                const uint32_t* orig = nullptr, unsigned long long* hash_out = nullptr) {
  /* the opt-in to > 48 KB of dynamic shared memory is a per-device function attribute: set it on every launch (a
     host-side call of about a microsecond) rather than once per process, so that contexts on several devices work */
  cudaFuncSetAttribute(pair_mma_kernel<Op, MC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)PairCfg<Op>::SMEM);
  pair_mma_kernel<Op, MC><<<(int)((N + BH - 1) / BH), PT, PairCfg<Op>::SMEM, st>>>(N, kp, grid, so, rec, orig, hash_out);
  return 1;
}

template <int D>
void launch_smoothing(int64_t N, const KParams& kp, const Grid* grid, const Sorted& so, cudaStream_t st) {
  launch_pair<SmoothOp<D>, 1>(N, kp, grid, so, so.rec_s, st);
}

/* test hook: the smoothing pass once more with the neighbour-set hash (no mask cache involved) */
template <int D>
void launch_smoothing_hash(int64_t N, const KParams& kp, const Grid* grid, const Sorted& so, const uint32_t* orig,
                           unsigned long long* hash_out, cudaStream_t st) {
  launch_pair<SmoothOp<D, true>, 0>(N, kp, grid, so, so.rec_s, st, orig, hash_out);
}

template <int D>
void launch_gradient(int64_t N, const KParams& kp, const Grid* grid, const Sorted& so, bool visc, bool diff, cudaStream_t st) {
  if (visc && diff) launch_pair<GradOp<D, true, true>, 2>(N, kp, grid, so, so.rec_g, st);
  else if (visc) launch_pair<GradOp<D, true, false>, 2>(N, kp, grid, so, so.rec_g, st);
  else if (diff) launch_pair<GradOp<D, false, true>, 2>(N, kp, grid, so, so.rec_g, st);
  else launch_pair<GradOp<D, false, false>, 2>(N, kp, grid, so, so.rec_g, st);
}

template <int D>
void launch_eps_gradient(int64_t N, const KParams& kp, const Grid* grid, const Sorted& so, cudaStream_t st) {
  launch_pair<EpsGradOp<D>, 2>(N, kp, grid, so, so.rec_s, st);
}

}  // namespace ccake
