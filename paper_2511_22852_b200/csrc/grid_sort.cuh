/*
 * csrc/grid_sort.cuh — steps a1-a3: bounding box, cell hash, stable LSD radix sort by cell, cell lists.
 * PAPER.md :1434 (§5.9.1): "particles are spatially binned ... neighbours drawn from nearby cells within a
 * cut-off radius", O(N).  Integer work only, except the fp64 coordinate -> cell index map, which uses
 * round-to-nearest multiplies without FMA contraction so that the reported cell ids are reproducible bit by bit.
 */
#pragma once
#include "common.cuh"

namespace ccake {

constexpr int BBOX_THREADS = 256;
constexpr int SORT_THREADS = 256;
constexpr int SORT_ITEMS = 16;
constexpr int SORT_TILE = SORT_THREADS * SORT_ITEMS;
constexpr int SCAN_CHUNK = 1024;

/* ------------------------------------------------------------------------------------------- a1 bbox ---- */
__device__ inline double warp_min(double v) {
  for (int o = 16; o > 0; o >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
__device__ inline double warp_max(double v) {
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

/* the threads of ONE block (at least 6 warps): reduce the partials (min/max are exact and order-free) and lay out the
   traversal grid */
__device__ __forceinline__ void bbox_finish(const double* partial, int nblocks, int D, double h, int max_cells, Grid* __restrict__ grid) {
  __shared__ double red[6];
  if (threadIdx.x < 192) {
    /* warp q reduces quantity q (0..2: minima, 3..5: maxima), its lanes striding over the blocks */
    const int q = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double r = __ldcg(partial + q);                    /* written by other blocks of this launch */
    for (int b = lane; b < nblocks; b += 32) {
      const double v = __ldcg(partial + b * 6 + q);
      r = (q < 3) ? fmin(r, v) : fmax(r, v);
    }
    for (int o = 16; o > 0; o >>= 1) {
      const double v = __shfl_xor_sync(0xffffffffu, r, o);
      r = (q < 3) ? fmin(r, v) : fmax(r, v);
    }
    if (lane == 0) red[q] = r;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    Grid g;
    for (int k = 0; k < 3; ++k) {
      g.xmin[k] = (k < D) ? red[k] : 0.0;
      g.xmax[k] = (k < D) ? red[3 + k] : 0.0;
    }
    const double twoh = 2.0 * h;
    double edge = twoh * GRID_MARGIN;
    /* coarsen by powers of two until the cell count fits the radix-sort key width chosen at load time */
    for (int it = 0; it < 64; ++it) {
      double total = 1.0;
      for (int k = 0; k < 3; ++k) {
        g.nc[k] = 1;
        if (k < D) {
          double ext = (g.xmax[k] - g.xmin[k]) / edge;
          if (!(ext >= 0.0)) ext = 0.0;
          if (ext > 1.0e9) ext = 1.0e9;
          g.nc[k] = (int)floor(ext) + 1;
        }
        total *= (double)g.nc[k];
      }
      if (total <= (double)max_cells) break;
      edge *= 2.0;
    }
    g.edge = edge;
    g.inv_edge = 1.0 / edge;
    g.ncells = g.nc[0] * g.nc[1] * g.nc[2];
    g.rep_inv_edge = 1.0 / twoh;
    g.mb = (D == 3) ? 9 : 8;
    {
      double ext = 0.0;
      for (int k = 0; k < D; ++k) ext = fmax(ext, g.xmax[k] - g.xmin[k]);
      if (!(ext < 1.0e300)) ext = 1.0e300;
      g.cutm = twoh + ext * (1.0 / 1048576.0);                       /* 2^-20 of the extent >> FP32 rounding 2^-24 */
      g.cutm2 = __double2float_ru(g.cutm * g.cutm * (1.0 + 1.0e-5));
    }
    for (int k = 0; k < 3; ++k) {
      g.rep_nc[k] = 1;
      if (k < D) g.rep_nc[k] = (long long)floor(__dmul_rn(__dsub_rn(g.xmax[k], g.xmin[k]), g.rep_inv_edge)) + 1;
    }
    *grid = g;
  }
}

/* partial[block][0..5] = min x,y,z, max x,y,z over the block's grid-stride share; the block that finishes last (a ticket
   counter, left at 0 for the next launch) reduces the partials and writes the grid: one launch for step a1 */
__global__ void __launch_bounds__(BBOX_THREADS)
bbox_kernel(const double* __restrict__ Y, int64_t npad, int64_t n, int D, double* partial, unsigned int* __restrict__ ticket,
            double h, int max_cells, Grid* __restrict__ grid) {
  double lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    for (int k = 0; k < 3; ++k) {
      if (k < D) {
        const double v = Y[(CCAKE_R1 + k) * npad + i];
        lo[k] = fmin(lo[k], v);
        hi[k] = fmax(hi[k], v);
      }
    }
  }
  __shared__ double sm[6][BBOX_THREADS / 32];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  for (int k = 0; k < 3; ++k) {
    const double a = warp_min(lo[k]), b = warp_max(hi[k]);
    if (lane == 0) { sm[k][w] = a; sm[3 + k][w] = b; }
  }
  __syncthreads();
  if (threadIdx.x < 6) {
    double r = sm[threadIdx.x][0];
    for (int j = 1; j < BBOX_THREADS / 32; ++j) r = (threadIdx.x < 3) ? fmin(r, sm[threadIdx.x][j]) : fmax(r, sm[threadIdx.x][j]);
    partial[blockIdx.x * 6 + threadIdx.x] = r;
  }
  __shared__ bool last;
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) {
    last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    if (last) *ticket = 0u;
  }
  __syncthreads();
  if (!last) return;
  __threadfence();
  bbox_finish(partial, (int)gridDim.x, D, h, max_cells, grid);
}

/* ------------------------------------------------------------------------------------------ a2 hash ---- */
__device__ inline int cell_coord(double x, double xmin, double inv_edge, int nc) {
  const double t = floor(__dmul_rn(__dsub_rn(x, xmin), inv_edge));
  int c = 0;
  if (t >= 0.0) c = (t < (double)nc) ? (int)t : nc - 1;   /* NaN -> 0 */
  return c;
}

/* Hilbert index of the sub-cell (X[0..D-1], nb bits each): Skilling's transpose algorithm ("Programming the
   Hilbert curve", 2004) followed by the bit interleave.  The curve visits every sub-cell once, consecutive
   indices are face neighbours, and it runs from corner (0,..,0) to corner (max,0,..,0) — so with cells ordered x
   fastest it continues into the next cell of the row without a jump.  Any bijection would be correct here;
   this one makes every run of consecutive sorted particles spatially compact, which is what the pair kernels'
   register tile (2 particles per thread, 2 threads per stream) needs. */
__device__ inline uint32_t hilbert_index(uint32_t* X, int nb, int D) {
  const uint32_t M = 1u << (nb - 1);
  for (uint32_t Q = M; Q > 1u; Q >>= 1) {
    const uint32_t P = Q - 1u;
    for (int i = 0; i < D; ++i) {
      if (X[i] & Q) X[0] ^= P;
      else { const uint32_t t = (X[0] ^ X[i]) & P; X[0] ^= t; X[i] ^= t; }
    }
  }
  for (int i = 1; i < D; ++i) X[i] ^= X[i - 1];
  uint32_t t = 0;
  for (uint32_t Q = M; Q > 1u; Q >>= 1)
    if (X[D - 1] & Q) t ^= Q - 1u;
  for (int i = 0; i < D; ++i) X[i] ^= t;
  uint32_t h = 0;
  for (int q = nb - 1; q >= 0; --q)
    for (int i = 0; i < D; ++i) h = (h << 1) | ((X[i] >> q) & 1u);
  return h;
}

/* sort key: traversal cell (x fastest) in the high bits; below it the Hilbert index of the position inside the
   cell (3 bits per axis in 3-D, 4 in 2-D), so that consecutive particles form compact clusters */
__global__ void cell_hash_kernel(const double* __restrict__ Y, int64_t npad, int64_t n, int D,
                                 const Grid* __restrict__ grid, uint32_t* __restrict__ key, uint32_t* __restrict__ val) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= n) return;
  const Grid g = *grid;
  int c[3] = {0, 0, 0};
  uint32_t sub3[3] = {0, 0, 0};
  const int sb = g.mb / D;               /* bits per axis */
  for (int k = 0; k < 3; ++k)
    if (k < D) {
      const double x = Y[(CCAKE_R1 + k) * npad + i];
      c[k] = cell_coord(x, g.xmin[k], g.inv_edge, g.nc[k]);
      const double frac = (x - g.xmin[k]) * g.inv_edge - (double)c[k];
      int sub = (int)(frac * (double)(1 << sb));
      sub3[k] = (uint32_t)max(0, min(sub, (1 << sb) - 1));
    }
  const int row = snake_row(g, c[1], c[2]);
  if (row & 1) sub3[0] = (uint32_t)((1 << sb) - 1) - sub3[0];      /* odd rows run backwards in x */
  const uint32_t morton = hilbert_index(sub3, sb, D);
  int cell_i, cell_last;
  snake_range(g, row, c[0], c[0], cell_i, cell_last);
  const uint32_t cell = (uint32_t)cell_i;
  key[i] = (cell << g.mb) | morton;
  val[i] = (uint32_t)i;
}

/* reported cell id (field CCAKE_CELL): edge exactly 2h, origin = exact coordinate minimum, product then floor */
__global__ void reported_cell_kernel(const double* __restrict__ x0, const double* __restrict__ x1,
                                     const double* __restrict__ x2, int64_t n, int D, const Grid* __restrict__ grid,
                                     double* __restrict__ out) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= n) return;
  const Grid g = *grid;
  const double* xs[3] = {x0, x1, x2};
  long long c[3] = {0, 0, 0};
  for (int k = 0; k < 3; ++k)
    if (k < D) c[k] = (long long)floor(__dmul_rn(__dsub_rn(xs[k][i], g.xmin[k]), g.rep_inv_edge));
  out[i] = (double)(c[0] + g.rep_nc[0] * (c[1] + g.rep_nc[1] * c[2]));
}

/* ------------------------------------------------------------------------------- a3 stable radix sort ---- */
/* pass 1 of 3: per-tile digit histogram; hist[d * ntiles + tile] */
__global__ void __launch_bounds__(SORT_THREADS)
radix_hist_kernel(const uint32_t* __restrict__ key, int64_t n, int shift, int ntiles, uint32_t* __restrict__ hist) {
  __shared__ uint32_t sh[256];
  sh[threadIdx.x] = 0;
  __syncthreads();
  const int64_t base = (int64_t)blockIdx.x * SORT_TILE;
  for (int r = 0; r < SORT_ITEMS; ++r) {
    const int64_t i = base + r * SORT_THREADS + threadIdx.x;
    if (i < n) atomicAdd(&sh[(key[i] >> shift) & 255u], 1u);
  }
  __syncthreads();
  hist[(int64_t)threadIdx.x * ntiles + blockIdx.x] = sh[threadIdx.x];
}

/* exclusive scan of m entries in chunks of SCAN_CHUNK: (1) in-chunk scan + chunk totals, (2) one block scans the
   totals, (3) consumers add chunk_off[idx / SCAN_CHUNK] */
__global__ void __launch_bounds__(SCAN_CHUNK)
scan_chunk_kernel(uint32_t* __restrict__ data, int64_t m, uint32_t* __restrict__ chunk_tot) {
  __shared__ uint32_t wsum[32];
  const int64_t i = (int64_t)blockIdx.x * SCAN_CHUNK + threadIdx.x;
  const uint32_t v = (i < m) ? data[i] : 0u;
  uint32_t x = v;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
    if (lane >= o) x += y;
  }
  if (lane == 31) wsum[w] = x;
  __syncthreads();
  if (w == 0) {
    uint32_t s = wsum[lane];
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t y = __shfl_up_sync(0xffffffffu, s, o);
      if (lane >= o) s += y;
    }
    wsum[lane] = s;
  }
  __syncthreads();
  const uint32_t incl = x + (w ? wsum[w - 1] : 0u);
  if (i < m) data[i] = incl - v;
  if (threadIdx.x == SCAN_CHUNK - 1) chunk_tot[blockIdx.x] = incl;
}

__global__ void __launch_bounds__(1024)
scan_totals_kernel(uint32_t* __restrict__ chunk_tot, int nchunks) {
  __shared__ uint32_t wsum[32];
  __shared__ uint32_t carry_s;
  if (threadIdx.x == 0) carry_s = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  for (int base = 0; base < nchunks; base += 1024) {
    const int i = base + threadIdx.x;
    const uint32_t v = (i < nchunks) ? chunk_tot[i] : 0u;
    uint32_t x = v;
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
      if (lane >= o) x += y;
    }
    if (lane == 31) wsum[w] = x;
    __syncthreads();
    if (w == 0) {
      uint32_t s = wsum[lane];
      for (int o = 1; o < 32; o <<= 1) {
        const uint32_t y = __shfl_up_sync(0xffffffffu, s, o);
        if (lane >= o) s += y;
      }
      wsum[lane] = s;
    }
    __syncthreads();
    const uint32_t incl = x + (w ? wsum[w - 1] : 0u) + carry_s;
    if (i < nchunks) chunk_tot[i] = incl - v;
    __syncthreads();
    if (threadIdx.x == 1023) carry_s = incl;
    __syncthreads();
  }
}

/* pass 3 of 3: stable scatter.  Keys of a tile are visited in rounds of SORT_THREADS consecutive keys; within a
   round the rank of a key among equal digits is (keys of earlier rounds) + (equal digits in lower warps) +
   (equal digits in lower lanes), which preserves the input order. */
__global__ void __launch_bounds__(SORT_THREADS, 4)
radix_scatter_kernel(const uint32_t* __restrict__ key_in, const uint32_t* __restrict__ val_in, int64_t n, int shift,
                     int ntiles, const uint32_t* __restrict__ hist, const uint32_t* __restrict__ chunk_off,
                     uint32_t* __restrict__ key_out, uint32_t* __restrict__ val_out) {
  constexpr int NW = SORT_THREADS / 32;
  __shared__ uint32_t wc[NW][256];
  __shared__ uint32_t run[256];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  {
    const int64_t hidx = (int64_t)threadIdx.x * ntiles + blockIdx.x;
    run[threadIdx.x] = hist[hidx] + chunk_off[hidx / SCAN_CHUNK];
    for (int j = 0; j < NW; ++j) wc[j][threadIdx.x] = 0;
  }
  __syncthreads();
  const int64_t base = (int64_t)blockIdx.x * SORT_TILE;
  /* all keys and values of the thread are loaded up front: one memory latency per tile instead of one per round */
  uint32_t kk[SORT_ITEMS], vv[SORT_ITEMS];
#pragma unroll
  for (int r = 0; r < SORT_ITEMS; ++r) {
    const int64_t i = base + r * SORT_THREADS + threadIdx.x;
    kk[r] = 0; vv[r] = 0;
    if (i < n) { kk[r] = key_in[i]; vv[r] = val_in[i]; }
  }
  const int rounds = (int)min((int64_t)SORT_ITEMS, (n - base + SORT_THREADS - 1) / SORT_THREADS);   /* the last tile may be short */
#pragma unroll
  for (int r = 0; r < SORT_ITEMS; ++r) {
    if (r >= rounds) break;
    const int64_t i = base + r * SORT_THREADS + threadIdx.x;
    const bool ok = i < n;
    const uint32_t k = kk[r], v = vv[r];
    const uint32_t d = ok ? ((k >> shift) & 255u) : 256u;
    const uint32_t mask = __match_any_sync(0xffffffffu, d);
    const uint32_t rank_w = __popc(mask & ((1u << lane) - 1u));
    if (ok && rank_w == 0) wc[w][d] = __popc(mask);
    __syncthreads();
    uint32_t pos = 0;
    if (ok) {
      pos = run[d] + rank_w;
      for (int j = 0; j < w; ++j) pos += wc[j][d];
    }
    __syncthreads();
    {
      uint32_t tot = 0;
      for (int j = 0; j < NW; ++j) { tot += wc[j][threadIdx.x]; wc[j][threadIdx.x] = 0; }
      run[threadIdx.x] += tot;
    }
    __syncthreads();
    if (ok) { key_out[pos] = k; val_out[pos] = v; }
  }
}

/* monotone cell_start[0..ncells]: cell c owns sorted slots [cell_start[c], cell_start[c+1]) */
__global__ void cell_start_kernel(const uint32_t* __restrict__ key, int64_t n, const Grid* __restrict__ grid,
                                  uint32_t* __restrict__ cell_start) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int mb = grid->mb;
  const int64_t k1 = key[i] >> mb;
  const int64_t k0 = (i == 0) ? -1 : (int64_t)(key[i - 1] >> mb);
  for (int64_t c = k0 + 1; c <= k1; ++c) cell_start[c] = (uint32_t)i;
  if (i == n - 1) {
    const int ncells = grid->ncells;
    for (int64_t c = k1 + 1; c <= ncells; ++c) cell_start[c] = (uint32_t)n;
  }
}

/* ------------------------------------------------------------------------------ reorder and pack ---- */
/* physical reorder of the store at the first substep of a step: dst[f][i] = src[f][perm[i]] for the active
   fields; afterwards the store order IS the sorted order and perm becomes the identity */
__global__ void reorder_store_kernel(const double* __restrict__ src, double* __restrict__ dst, int64_t npad, int64_t n,
                                     uint32_t* __restrict__ perm, uint32_t field_mask,
                                     const uint32_t* __restrict__ orig_src, uint32_t* __restrict__ orig_dst) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint32_t a = perm[i];
  for (int f = 0; f < NSTATE; ++f)
    if (field_mask & (1u << f)) dst[f * npad + i] = src[f * npad + a];
  orig_dst[i] = orig_src[a];
  perm[i] = (uint32_t)i;           /* entry i is read by this thread only */
}

__global__ void iota_kernel(uint32_t* __restrict__ p, int64_t n) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i < n) p[i] = (uint32_t)i;
}

/* sorted order: exact positions, FP32 positions relative to the grid origin (culling only), and the AoS payload
   record of the smoothing pass: x[3], m, S, N_B, N_S, N_Q */
__global__ void pack_smoothing_kernel(const double* __restrict__ Y, int64_t npad, int64_t n, int D,
                                      const uint32_t* __restrict__ perm, const Grid* __restrict__ grid, Sorted so) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint32_t a = perm[i];
  const double x = Y[CCAKE_R1 * npad + a], y = Y[CCAKE_R2 * npad + a], z = (D == 3) ? Y[CCAKE_R3 * npad + a] : 0.0;
  so.x[0][i] = x; so.x[1][i] = y; so.x[2][i] = z;
  so.xf[i] = make_float4((float)(x - grid->xmin[0]), (float)(y - grid->xmin[1]), (D == 3) ? (float)(z - grid->xmin[2]) : 0.f,
                         __uint_as_float((uint32_t)i));   /* w: the sorted slot (read by the neighbour-hash test pass) */
  const double m = Y[CCAKE_MASS * npad + a];              /* payload columns carry the SPH weight m_b (pair_mma.cuh) */
  double* r = so.rec_s + i * 8;                           /* 64-byte record: two 32-byte stores (STG.256) */
  asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(r), "d"(x), "d"(y), "d"(z), "d"(m) : "memory");
  asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(r + 4), "d"(m * Y[CCAKE_S * npad + a]), "d"(m * Y[CCAKE_NB * npad + a]),
               "d"(m * Y[CCAKE_NS * npad + a]), "d"(m * Y[CCAKE_NQ * npad + a]) : "memory");
}

}  // namespace ccake
