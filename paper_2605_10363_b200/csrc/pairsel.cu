// Executable-pair selection for the rho contraction (Eq. 17-19), run per call because the
// block summary b_qr = max|D_qr| of the second operand changes with D (reading A6 of DESIGN.md):
//   k_dmax        b_qr for every AO-shell pair of the plan-order density matrix (Eq. 11 applied to D);
//   k_pair_select for every grid block p the set of (32-column K chunk, N tile) stages of k_rho that contain at
//                 least one executable pair a_pq * b_qr >= t_d (Eq. 17, 19); a stage without one is skipped.
// The skippable unit of this design is a ring stage, not a single block pair: the retained columns of a grid
// block are packed in spatial (plan) order, so a chunk is a compact group of ~2 molecules and a tile ~6-8, and a
// localised D empties whole (chunk, tile) stages.  Alg. 1's mask + prefix-sum compaction is the
// 64-bit mask per grid block written here and scanned by the producer warps.
#include "kldi_internal.h"

namespace kldi {

// One thread per shell pair (q, r), plan order.  tri: Dp holds the lower triangle with the diagonal halved
// (k_permute_D<true>), only q >= r is needed and the halved diagonal is doubled back (conservative).
__global__ void __launch_bounds__(128) k_dmax(const double* __restrict__ Dp, int n_ao, int n_shells,
                                              const int32_t* __restrict__ sh_ao0, int tri, double* __restrict__ b) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x, q = blockIdx.y;
  if (r >= n_shells || (tri && r > q)) return;
  const int i0 = sh_ao0[q], i1 = sh_ao0[q + 1], j0 = sh_ao0[r], j1 = sh_ao0[r + 1];
  double m = 0.0;
  for (int i = i0; i < i1; ++i)
    for (int j = j0; j < j1; ++j) {
      if (tri && j > i) continue;
      double v = fabs(Dp[(int64_t)i * n_ao + j]);
      if (tri && i == j) v *= 2.0;
      m = fmax(m, v);
    }
  b[(int64_t)q * n_shells + r] = m;
}

// One warp per non-empty grid block.  mask bit (k0/32)*4 + jt <=> stage (chunk k0, tile jt) has an executable pair.
// Panels with more than 16 chunks or 4 tiles keep every stage (mask = all ones).
__global__ void __launch_bounds__(128) k_pair_select(const int32_t* __restrict__ tasks, int n_tasks,
                                                     const int32_t* __restrict__ row_ptr,
                                                     const int32_t* __restrict__ col_idx,
                                                     const int32_t* __restrict__ blk_col0,
                                                     const int32_t* __restrict__ sh_ao0,
                                                     const double* __restrict__ amax, const int32_t* __restrict__ kp,
                                                     const double* __restrict__ b, int n_shells, double eps, int tri,
                                                     unsigned long long* __restrict__ mask,
                                                     unsigned long long* __restrict__ counters) {
  const int lane = threadIdx.x & 31;
  const int t = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (t >= n_tasks) return;
  const int p = tasks[t];
  const int K8 = (kp[p] + 7) & ~7;
  const int ntile = (K8 + 127) / 128;
  const int W = tri ? (((K8 + ntile - 1) / ntile) + 31) & ~31 : (((K8 + ntile - 1) / ntile) + 7) & ~7;
  const int nchunk = (K8 + 31) / 32;
  unsigned long long m = 0ull, all = 0ull;
  for (int jt = 0; jt < ntile; ++jt)  // the stages k_rho would run without the test
    for (int c = tri ? (jt * W) / 32 : 0; c < nchunk; ++c) all |= 1ull << ((c & 15) * 4 + (jt & 3));
  if (nchunk > 16 || ntile > 4 || eps <= 0.0) {
    if (lane == 0) mask[p] = ~0ull;
    return;
  }
  const int e0 = row_ptr[p], ne = row_ptr[p + 1] - e0;
  for (int qi = 0; qi < ne; ++qi) {
    const int sq = col_idx[e0 + qi], cq0 = blk_col0[e0 + qi], wq = sh_ao0[sq + 1] - sh_ao0[sq];
    const double aq = amax[e0 + qi];
    const int ch0 = cq0 >> 5, ch1 = (cq0 + wq - 1) >> 5;
    for (int ri = lane; ri < (tri ? qi + 1 : ne); ri += 32) {
      const int sr = col_idx[e0 + ri];
      // Eq. 17: retain iff a_pq b_qr >= t_d.  In the triangular form one stage stands for both orientations (q,r) and
      // (r,q) of the symmetric D, so it runs if EITHER is executable: max(a_pq, a_pr) b_qr >= t_d (a conservative superset)
      const double aa = tri ? fmax(aq, amax[e0 + ri]) : aq;
      if (aa * b[(int64_t)sq * n_shells + sr] >= eps) {
        const int cr0 = blk_col0[e0 + ri], wr = sh_ao0[sr + 1] - sh_ao0[sr];
        for (int jt = cr0 / W; jt <= (cr0 + wr - 1) / W; ++jt)
          for (int c = ch0; c <= ch1; ++c) m |= 1ull << (c * 4 + jt);
      }
    }
  }
  for (int o = 16; o > 0; o >>= 1) m |= __shfl_xor_sync(0xffffffffu, m, o);
  if (lane == 0) {
    mask[p] = m;
    atomicAdd(counters, (unsigned long long)__popcll(all));
    atomicAdd(counters + 1, (unsigned long long)__popcll(m & all));
  }
}

kldi_status launch_pair_select(kldi_plan* P, bool tri) {
  const size_t nb = sizeof(double) * (size_t)P->n_shells * P->n_shells;
  if (!P->d_bmax) KLDI_CUDA(cudaMalloc(&P->d_bmax, nb));
  if (!P->d_pmask) {
    KLDI_CUDA(cudaMalloc(&P->d_pmask, sizeof(unsigned long long) * (size_t)(P->n_blocks + 2)));
    P->d_pcount = P->d_pmask + P->n_blocks;
  }
  KLDI_CUDA(cudaMemsetAsync(P->d_pcount, 0, 2 * sizeof(unsigned long long), P->stream));
  if (P->n_tasks == 0) return KLDI_OK;
  dim3 g((P->n_shells + 127) / 128, P->n_shells);
  k_dmax<<<g, 128, 0, P->stream>>>(P->d_Dp, P->n_ao, P->n_shells, P->d_sh_ao0, tri ? 1 : 0, P->d_bmax);
  KLDI_LAUNCHED(P);
  k_pair_select<<<(P->n_tasks + 3) / 4, 128, 0, P->stream>>>(
      P->d_tasks, P->n_tasks, P->d_row_ptr, P->d_col_idx, P->d_blk_col0, P->d_sh_ao0, P->d_blk_amax, P->d_kp,
      P->d_bmax, P->n_shells, P->eps, tri ? 1 : 0, P->d_pmask, P->d_pcount);
  KLDI_LAUNCHED(P);
  P->pair_counts_valid = true;
  return KLDI_OK;
}

}  // namespace kldi
