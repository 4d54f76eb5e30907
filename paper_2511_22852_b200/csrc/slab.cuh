/*
 * csrc/slab.cuh — slab decomposition of ONE event over several contexts (not in the paper, which
 * runs one event per device): device kernels that select, pack and unpack the particles that cross a slab face.
 *
 * A slab context owns the particles with lo <= r[axis] < hi and carries, behind them in load order, GHOST copies of the
 * neighbours' particles within W of its faces.  W covers two kernel supports (4h) plus the drift of a step, so that with
 * ONE exchange of particle states per substep every owned particle sees complete neighbours twice over: its smoothing
 * sums (neighbours within 2h) and, for its gradient sums, the smoothing sums and thermodynamics of those neighbours
 * (their neighbours within another 2h), which the context recomputes for its ghosts.  Ghost rates are not valid and are
 * never used: the ghost states are re-imported before every substep.
 *
 *   step:  export_halo(k = 0) -> import_ghosts(k = 0) -> substep 0 -> [ export_halo(k) -> import_ghosts(k) -> substep k ] ...
 *          -> export_migrants -> import_migrants -> commit (owned set rebuilt: stayers in store order, then arrivals)
 *
 * With NARROW halos (W = 2h + drift) the ghosts' own sums are incomplete; then the gradient records of the halo particles
 * travel as a second message between a5 and a6 (substep_a -> export_records -> import_records -> substep_b): half the ghosts,
 * twice the messages.
 *
 * Exchange buffers (device memory of the caller, moved by the caller's transport: a device copy, or NCCL send/recv):
 * SLAB_NF rows of `cap` doubles, row f < NSTATE = state field f, row NSTATE = the global particle id; entry i of
 * every row belongs to particle i of the message.  Selection is by flags + exclusive scan (grid_sort.cuh), so the order
 * of a message is the store order of the sender: deterministic, no atomics.
 */
#pragma once
#include "common.cuh"
#include "grid_sort.cuh"

namespace ccake {

constexpr int SLAB_NF = NSTATE + 1;

/* class of store slot a at the end of a step / for the halo of a step: 0 stays (or is not selected), 1 low side, 2 high side,
   3 ghost (dropped) */
__device__ __forceinline__ int slab_class(const double* __restrict__ Y, int64_t npad, int64_t a, int axis, double lo_edge,
                                          double hi_edge, const uint32_t* __restrict__ orig, int64_t n_own) {
  if ((int64_t)orig[a] >= n_own) return 3;
  const double x = Y[(CCAKE_R1 + axis) * npad + a];
  if (x < lo_edge) return 1;
  if (x >= hi_edge) return 2;
  return 0;
}

/* flags of the three classes that are kept (0 stay, 1 low, 2 high); a NULL array is skipped */
__global__ void slab_flag_kernel(const double* __restrict__ Y, int64_t npad, int64_t n, int axis, double lo_edge, double hi_edge,
                                 const uint32_t* __restrict__ orig, int64_t n_own, uint32_t* __restrict__ f_stay,
                                 uint32_t* __restrict__ f_lo, uint32_t* __restrict__ f_hi) {
  const int64_t a = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (a >= n) return;
  const int c = slab_class(Y, npad, a, axis, lo_edge, hi_edge, orig, n_own);
  if (f_stay) f_stay[a] = (c == 0) ? 1u : 0u;
  if (f_lo) f_lo[a] = (c == 1) ? 1u : 0u;
  if (f_hi) f_hi[a] = (c == 2) ? 1u : 0u;
}

/* number of selected entries after the two scan kernels: rank of the last slot + its own flag */
__global__ void slab_count_kernel(const uint32_t* __restrict__ rank, const uint32_t* __restrict__ chunk_off, int64_t n,
                                  const double* __restrict__ Y, int64_t npad, int axis, double lo_edge, double hi_edge,
                                  const uint32_t* __restrict__ orig, int64_t n_own, int cls, long long* __restrict__ out) {
  if (n <= 0) { *out = 0; return; }
  const int64_t a = n - 1;
  const int c = slab_class(Y, npad, a, axis, lo_edge, hi_edge, orig, n_own);
  *out = (long long)rank[a] + (long long)chunk_off[a / SCAN_CHUNK] + ((c == cls) ? 1 : 0);
}

/* message of class cls: all state fields + global id, in store order; list (may be NULL) = load indices of the entries */
__global__ void slab_pack_kernel(const double* __restrict__ Y, int64_t npad, int64_t n, int axis, double lo_edge, double hi_edge,
                                 const uint32_t* __restrict__ orig, int64_t n_own, int cls, const uint32_t* __restrict__ rank,
                                 const uint32_t* __restrict__ chunk_off, const uint32_t* __restrict__ gid, double* __restrict__ buf,
                                 int64_t cap, uint32_t* __restrict__ list) {
  const int64_t a = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (a >= n) return;
  if (slab_class(Y, npad, a, axis, lo_edge, hi_edge, orig, n_own) != cls) return;
  const int64_t r = (int64_t)rank[a] + chunk_off[a / SCAN_CHUNK];
  if (r >= cap) return;                                   /* the host reports the overflow from the count */
#pragma unroll 4
  for (int f = 0; f < NSTATE; ++f) buf[(int64_t)f * cap + r] = Y[(int64_t)f * npad + a];
  buf[(int64_t)NSTATE * cap + r] = (double)gid[orig[a]];
  if (list) list[r] = orig[a];
}

/* the same particles once more (later substeps): entry i = load index list[i], read from the stage state */
__global__ void slab_repack_kernel(const double* __restrict__ Y, int64_t npad, int64_t cnt, const uint32_t* __restrict__ list,
                                   const uint32_t* __restrict__ slot_of, const uint32_t* __restrict__ gid, double* __restrict__ buf,
                                   int64_t cap) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= cnt) return;
  const uint32_t li = list[i];
  const int64_t a = slot_of[li];
#pragma unroll 4
  for (int f = 0; f < NSTATE; ++f) buf[(int64_t)f * cap + i] = Y[(int64_t)f * npad + a];
  buf[(int64_t)NSTATE * cap + i] = (double)gid[li];
}

/* ghosts of a new step: appended behind the current particles, load indices load0 + i */
__global__ void slab_append_kernel(double* __restrict__ Y, int64_t npad, int64_t slot0, int64_t load0, int64_t cnt,
                                   const double* __restrict__ buf, int64_t cap, uint32_t* __restrict__ orig, uint32_t* __restrict__ gid) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= cnt) return;
#pragma unroll 4
  for (int f = 0; f < NSTATE; ++f) Y[(int64_t)f * npad + slot0 + i] = buf[(int64_t)f * cap + i];
  orig[slot0 + i] = (uint32_t)(load0 + i);
  gid[load0 + i] = (uint32_t)buf[(int64_t)NSTATE * cap + i];
}

/* ghosts of a later substep: the stage state of load indices load0 + i is overwritten with the owner's */
__global__ void slab_refresh_kernel(double* __restrict__ Y, int64_t npad, int64_t load0, int64_t cnt, const double* __restrict__ buf,
                                    int64_t cap, const uint32_t* __restrict__ slot_of) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= cnt) return;
  const int64_t a = slot_of[load0 + i];
#pragma unroll 4
  for (int f = 0; f < NSTATE; ++f) Y[(int64_t)f * npad + a] = buf[(int64_t)f * cap + i];
}

__global__ void slab_inverse_kernel(const uint32_t* __restrict__ orig, int64_t n, uint32_t* __restrict__ slot_of) {
  const int64_t a = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (a < n) slot_of[orig[a]] = (uint32_t)a;
}

/* commit, part 1: the particles that stay, compacted in store order into the other state buffer */
__global__ void slab_keep_kernel(const double* __restrict__ Y, double* __restrict__ Ynew, int64_t npad, int64_t n, int axis,
                                 double lo, double hi, const uint32_t* __restrict__ orig, int64_t n_own,
                                 const uint32_t* __restrict__ rank, const uint32_t* __restrict__ chunk_off,
                                 const uint32_t* __restrict__ gid, uint32_t* __restrict__ gid_new) {
  const int64_t a = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (a >= n) return;
  if (slab_class(Y, npad, a, axis, lo, hi, orig, n_own) != 0) return;
  const int64_t r = (int64_t)rank[a] + chunk_off[a / SCAN_CHUNK];
#pragma unroll 4
  for (int f = 0; f < NSTATE; ++f) Ynew[(int64_t)f * npad + r] = Y[(int64_t)f * npad + a];
  gid_new[r] = gid[orig[a]];
}

/* commit, part 2: arrivals (parked messages) behind the stayers */
__global__ void slab_arrive_kernel(double* __restrict__ Ynew, int64_t npad, int64_t slot0, int64_t cnt, const double* __restrict__ buf,
                                   int64_t cap, int64_t col0, uint32_t* __restrict__ gid_new) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= cnt) return;
#pragma unroll 4
  for (int f = 0; f < NSTATE; ++f) Ynew[(int64_t)f * npad + slot0 + i] = buf[(int64_t)f * cap + col0 + i];
  gid_new[slot0 + i] = (uint32_t)buf[(int64_t)NSTATE * cap + col0 + i];
}

/* parked copy of an incoming migrant message */
__global__ void slab_park_kernel(const double* __restrict__ in, int64_t cap_in, int64_t cnt, double* __restrict__ park, int64_t cap,
                                 int64_t col0) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= cnt) return;
#pragma unroll 4
  for (int f = 0; f < SLAB_NF; ++f) park[(int64_t)f * cap + col0 + i] = in[(int64_t)f * cap_in + i];
}

/* ---- narrow halos: the gradient records of the halo particles travel between a5 and a6 ---- */
/* sorted slot of a store slot (inverse of perm) */
__global__ void slab_inverse_perm_kernel(const uint32_t* __restrict__ perm, int64_t n, uint32_t* __restrict__ sorted_of) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i < n) sorted_of[perm[i]] = (uint32_t)i;
}

/* message: nrec rows of cap doubles, entry i = the record of load index list[i] (the halo list of this step) */
__global__ void slab_pack_records_kernel(const double* __restrict__ rec, int nrec, int64_t cnt, const uint32_t* __restrict__ list,
                                         const uint32_t* __restrict__ slot_of, const uint32_t* __restrict__ sorted_of,
                                         double* __restrict__ buf, int64_t cap) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= cnt) return;
  const double* __restrict__ r = rec + (int64_t)sorted_of[slot_of[list[i]]] * nrec;
  for (int f = 0; f < nrec; ++f) buf[(int64_t)f * cap + i] = r[f];
}

/* the records of the ghosts with load indices load0 + i are overwritten with their owners' */
__global__ void slab_unpack_records_kernel(double* __restrict__ rec, int nrec, int64_t load0, int64_t cnt, const double* __restrict__ buf,
                                           int64_t cap, const uint32_t* __restrict__ slot_of, const uint32_t* __restrict__ sorted_of) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= cnt) return;
  double* __restrict__ r = rec + (int64_t)sorted_of[slot_of[load0 + i]] * nrec;
  for (int f = 0; f < nrec; ++f) r[f] = buf[(int64_t)f * cap + i];
}

__global__ void slab_iota_gid_kernel(uint32_t* __restrict__ gid, int64_t n, uint32_t base) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i < n) gid[i] = base + (uint32_t)i;
}

}  // namespace ccake
