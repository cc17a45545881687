// H4: V contraction.  Per grid block p the packed Gram matrix G_p = Phi_p^T diag(wv_p) Phi_p (LDA: strips
// on and above the diagonal; GGA: B_p = Phi_p^T Z_p, the full square) is formed by FP64 tensor-core MMAs
// (DMMA.8x8x4) and added to V (Eq. 5/16; accumulate-before-write-back).
// Persistent, warp-specialised: a producer warp pulls grid blocks from an atomic ticket (on
// device) and streams 32-row chunks of the panel columns a pass needs through a 3-stage mbarrier ring with
// bulk-async copies (TMA engine, SASS UBLKCP); V_WARPS (15) consumer warps each hold up to V_SLOTS (2)
// register-resident items (16 rows x <= 32 columns) chosen by the host schedule of vsched.h, so that ragged K_p
// keeps every warp busy.
#include <cstring>

#include "kldi_internal.h"
#include "ptx.cuh"
#include "vsched.h"

namespace kldi {

namespace vg {
constexpr int NST = V_SLAB == 16 ? 6 : 3;
constexpr int RC = V_SLAB;              // grid rows (the MMA K dimension) per ring stage = one slab of the V layout
constexpr int STR = RC;             // column stride in doubles: dense, the chunk swizzle of vlayout_off avoids conflicts
constexpr int NCOL = V_MAXCOLS + 8; // column slots per stage (+8: second row block of an odd last strip)
constexpr int COLS_BYTES = NCOL * STR * 8;
constexpr int IDX_OFF = COLS_BYTES + RC * 8;      // plan AO index of every staged column (for the epilogue)
constexpr int ITEM_OFF = IDX_OFF + ((NCOL * 4 + 127) / 128) * 128;     // the pass's 32 VItems (first slab only)
constexpr int STAGE_BYTES = ITEM_OFF + ((V_ITEMS * 8 + 127) / 128) * 128;          // columns + wv chunk + column indices + items
constexpr int SMEM_BYTES = NST * STAGE_BYTES + NST * 16 + 2 * NST * 8;
enum { F_FIRST = 1, F_LAST = 2, F_DONE = 4 };
}  // namespace vg

// One slab (32 grid rows = 8 k-steps) of one item.  A, B point at the item's first column (+ q4 columns);
// o0/o1 are the lane's swizzled offsets of chunks 2 r4 and 2 r4 + 1; a 16-byte load feeds two k-steps.
// DIAG: the item's first block sits on the diagonal of an LDA strip; its rows 8..15 lie strictly below it and are
// skipped (acc[1][0] stays zero and is never written back).
template <int NJ, bool GGA, bool DIAG>
__device__ __forceinline__ void vg_run(double (&acc)[2][4][2], const double* __restrict__ A,
                                       const double* __restrict__ B, const double* __restrict__ w, int o0, int o1) {
  using namespace vg;
#pragma unroll
  for (int h = 0; h < RC / 16; ++h) {
#pragma unroll
    for (int j = 0; j < 2; ++j) {
      const int o = (j ? o1 : o0) + 16 * h;
      double2 a0 = *reinterpret_cast<const double2*>(A + o);
      double2 a1 = *reinterpret_cast<const double2*>(A + 8 * STR + o);
      if (!GGA) {
        const double2 ww = *reinterpret_cast<const double2*>(w + 2 * j + 16 * h);
        a0.x *= ww.x; a0.y *= ww.y;
        a1.x *= ww.x; a1.y *= ww.y;
      }
      double2 b[NJ];
#pragma unroll
      for (int n = 0; n < NJ; ++n) b[n] = *reinterpret_cast<const double2*>(B + n * 8 * STR + o);
#pragma unroll
      for (int n = 0; n < NJ; ++n) {
        dmma884(acc[0][n][0], acc[0][n][1], a0.x, b[n].x);
        if (!(DIAG && n == 0)) dmma884(acc[1][n][0], acc[1][n][1], a1.x, b[n].x);
      }
#pragma unroll
      for (int n = 0; n < NJ; ++n) {
        dmma884(acc[0][n][0], acc[0][n][1], a0.y, b[n].y);
        if (!(DIAG && n == 0)) dmma884(acc[1][n][0], acc[1][n][1], a1.y, b[n].y);
      }
    }
  }
}

// EPI = 0: the epilogue adds G_p straight into the plan-order V with red.global.add.f64.
// EPI = 1: G_p goes to the workspace (plain 16-B stores) and k_vreduce sums it in a fixed order.
// EPI = 2: as 0, but in 64-bit fixed point with integer atomics: integer addition is associative, so V is bitwise
//          reproducible whatever the order of the adds; the scale is the power of two that keeps every partial sum
//          below 2^61 (k_fx_bound), the only rounding is that of a contribution to 2^-61 of the bound.
template <bool GGA, int EPI>
__global__ void __launch_bounds__(32 * (V_WARPS + 1), 1)
    k_vgram(const int32_t* __restrict__ tasks, int n_tasks, int32_t* __restrict__ ticket,
            const int32_t* __restrict__ kp, const int64_t* __restrict__ panel_off, const int32_t* __restrict__ colidx,
            const double* __restrict__ phi, const double* __restrict__ zmat, const double* __restrict__ wv_s,
            const int32_t* __restrict__ sched_ptr, const VPass* __restrict__ passes, const VItem* __restrict__ items,
            int n_ao, double* __restrict__ Vp, const int64_t* __restrict__ gram_off, double* __restrict__ G,
            const double* __restrict__ fx_bound) {
  using namespace vg;
  constexpr bool ATOMIC = (EPI != 1);
  extern __shared__ __align__(128) unsigned char smem[];
  int* hdr = reinterpret_cast<int*>(smem + NST * STAGE_BYTES);
  const uint32_t bar0 = smem_u32(smem + NST * STAGE_BYTES + NST * 16);  // full[s] at +8s, empty[s] at +8(NST+s)
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid == 0) {
    for (int s = 0; s < NST; ++s) {
      mbar_init(bar0 + 8 * s, 1);
      mbar_init(bar0 + 8 * (NST + s), V_WARPS);
    }
    fence_mbar_init();
  }
  __syncthreads();

  if (warp == V_WARPS) {
    // ------------------------------------------------------------------ producer warp
    int s = 0;
    uint32_t ph = 0;
    for (;;) {
      int t = 0;
      if (lane == 0) t = atomicAdd(ticket, 1);
      t = __shfl_sync(0xffffffffu, t, 0);
      if (t >= n_tasks) break;
      const int p = tasks[t];
      const int K8 = (kp[p] + 7) & ~7;
      const int nb = K8 >> 3;
      const int64_t base = panel_off[p];
      for (int ps = sched_ptr[nb]; ps < sched_ptr[nb + 1]; ++ps) {
        const VPass P = passes[ps];
        for (int rc = 0; rc < GB / RC; ++rc) {
          mbar_wait(bar0 + 8 * (NST + s), ph ^ 1);
          const uint32_t full = bar0 + 8 * s;
          if (lane == 0) {
            hdr[4 * s + 0] = p;
            hdr[4 * s + 1] = ps;
            hdr[4 * s + 2] = (rc == 0 ? F_FIRST : 0) | (rc == GB / RC - 1 ? F_LAST : 0);
            hdr[4 * s + 3] = K8 | (kp[p] << 16);
            mbar_arrive_expect_tx(full, (uint32_t)((P.c1_n + P.c2_n) * (RC * 8) + (GGA ? 0 : RC * 8) +
                                                   ((ATOMIC && rc == GB / RC - 1) ? (P.c1_n + P.c2_n) * 4 : 0) +
                                                   (rc == 0 ? V_ITEMS * 8 : 0)));
          }
          __syncwarp();
          if (lane == 0) {  // one bulk copy per column interval: the slab is contiguous in the V layout
            const uint32_t sa = smem_u32(smem + s * STAGE_BYTES);
            const int64_t slab = base * GB + (int64_t)rc * K8 * RC;
            bulk_g2s(sa, phi + slab + (int64_t)P.c1_lo * RC, (uint32_t)P.c1_n * (RC * 8), full);
            if (P.c2_n)
              bulk_g2s(sa + P.c1_n * (RC * 8), (GGA ? zmat : phi) + slab + (int64_t)P.c2_lo * RC,
                       (uint32_t)P.c2_n * (RC * 8), full);
            if (!GGA) bulk_g2s(sa + COLS_BYTES, wv_s + (int64_t)p * GB + rc * RC, RC * 8, full);
            if (rc == 0) bulk_g2s(sa + ITEM_OFF, items + (int64_t)ps * V_ITEMS, V_ITEMS * 8, full);
            if (ATOMIC && rc == GB / RC - 1) {  // last slab of the pass: column indices for the scatter epilogue
              bulk_g2s(sa + IDX_OFF, colidx + base + P.c1_lo, (uint32_t)P.c1_n * 4, full);
              if (P.c2_n) bulk_g2s(sa + IDX_OFF + P.c1_n * 4, colidx + base + P.c2_lo, (uint32_t)P.c2_n * 4, full);
            }
          }
          if (++s == NST) { s = 0; ph ^= 1; }
        }
      }
    }
    mbar_wait(bar0 + 8 * (NST + s), ph ^ 1);
    if (lane == 0) {
      hdr[4 * s + 2] = F_DONE;
      mbar_arrive(bar0 + 8 * s);
    }
    return;
  }

  // -------------------------------------------------------------------- consumer warps
  const int q4 = lane >> 2, r4 = lane & 3;
  const int o0 = ((2 * r4) ^ q4) * 2, o1 = ((2 * r4 + 1) ^ q4) * 2;  // swizzled chunk offsets (doubles)
  double acc[V_SLOTS][2][4][2];
  const double fxs = (EPI == 2) ? fx_scale(*fx_bound) : 1.0;
  int ia[V_SLOTS], ib[V_SLOTS];
#pragma unroll
  for (int k = 0; k < V_SLOTS; ++k) ia[k] = ib[k] = 0;
  int s = 0;
  uint32_t ph = 0;
  for (;;) {
    mbar_wait(bar0 + 8 * s, ph);
    const int p = hdr[4 * s + 0], fl = hdr[4 * s + 2];
    const int K8 = hdr[4 * s + 3] & 0xffff, K = hdr[4 * s + 3] >> 16;
    if (fl & F_DONE) break;
    if (fl & F_FIRST) {
      const VItem* it = reinterpret_cast<const VItem*>(smem + s * STAGE_BYTES + ITEM_OFF) + warp * V_SLOTS;
#pragma unroll
      for (int k = 0; k < V_SLOTS; ++k) {
        ia[k] = it[k].a;
        ib[k] = it[k].b;
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[k][0][j][0] = acc[k][0][j][1] = acc[k][1][j][0] = acc[k][1][j][1] = 0.0;
      }
    }
    const double* st = reinterpret_cast<const double*>(smem + s * STAGE_BYTES) + q4 * STR;
    const double* wb = reinterpret_cast<const double*>(smem + s * STAGE_BYTES + COLS_BYTES) + 4 * r4;
#pragma unroll
    for (int k = 0; k < V_SLOTS; ++k) {
      const double* A = st + (ia[k] & 1023) * STR;
      const double* B = st + ((ia[k] >> 10) & 1023) * STR;
      switch (ia[k] >> 20) {  // nj | diag << 4
        case 1: vg_run<1, GGA, false>(acc[k], A, B, wb, o0, o1); break;
        case 2: vg_run<2, GGA, false>(acc[k], A, B, wb, o0, o1); break;
        case 3: vg_run<3, GGA, false>(acc[k], A, B, wb, o0, o1); break;
        case 4: vg_run<4, GGA, false>(acc[k], A, B, wb, o0, o1); break;
        case 17: if (!GGA) vg_run<1, GGA, true>(acc[k], A, B, wb, o0, o1); break;
        case 18: if (!GGA) vg_run<2, GGA, true>(acc[k], A, B, wb, o0, o1); break;
        case 19: if (!GGA) vg_run<3, GGA, true>(acc[k], A, B, wb, o0, o1); break;
        case 20: if (!GGA) vg_run<4, GGA, true>(acc[k], A, B, wb, o0, o1); break;
        default: break;
      }
    }
    const int* sidx = reinterpret_cast<const int*>(smem + s * STAGE_BYTES + IDX_OFF);
    if (!(ATOMIC && (fl & F_LAST))) {  // the atomic epilogue still reads the stage's column indices
      __syncwarp();
      if (lane == 0) mbar_arrive(bar0 + 8 * (NST + s));
    }
    const int s_cur = s;
    if (++s == NST) { s = 0; ph ^= 1; }

    if (fl & F_LAST) {
#pragma unroll
      for (int k = 0; k < V_SLOTS; ++k) {
        const int nj = (ia[k] >> 20) & 7;
        if (nj == 0) continue;
        const int arow = ib[k] & 0xffff, bcol = ib[k] >> 16;
#pragma unroll
        for (int mi = 0; mi < 2; ++mi) {
          const int r = arow + 8 * mi + q4;
          if (ATOMIC) {
            if (r < K) {
              const int64_t ci = (int64_t)sidx[(ia[k] & 1023) + 8 * mi + q4] * n_ao;
              const int* cidx = sidx + ((ia[k] >> 10) & 1023) + 2 * r4;
#pragma unroll
              for (int j = 0; j < 4; ++j)
                if (j < nj) {
#pragma unroll
                  for (int e = 0; e < 2; ++e) {
                    const int c = bcol + 8 * j + 2 * r4 + e;
                    if (c < K && (GGA || r <= c)) {
                      if (EPI == 2)
                        atomicAdd(reinterpret_cast<unsigned long long*>(Vp) + ci + cidx[8 * j + e],
                                  (unsigned long long)__double2ll_rn(acc[k][mi][j][e] * fxs));
                      else
                        atomicAdd(Vp + ci + cidx[8 * j + e], acc[k][mi][j][e]);
                    }
                  }
                }
            }
          } else {
            if (arow + 8 * mi < K8) {
              // LDA: strip-packed upper triangle (strip s: 16 rows x (K8 - 16 s) columns); GGA: K8 x K8 square
              const int sx = arow >> 4;
              const int64_t rowoff = GGA ? (int64_t)r * K8
                                         : (int64_t)16 * sx * K8 - (int64_t)128 * sx * (sx - 1) +
                                               (int64_t)(8 * mi + q4) * (K8 - 16 * sx) - 16 * sx;
              double* g = G + gram_off[p] + rowoff + bcol + 2 * r4;
#pragma unroll
              for (int j = 0; j < 4; ++j)
                if (j < nj) *reinterpret_cast<double2*>(g + 8 * j) = make_double2(acc[k][mi][j][0], acc[k][mi][j][1]);
            }
          }
        }
      }
      if (ATOMIC) {
        __syncwarp();
        if (lane == 0) mbar_arrive(bar0 + 8 * (NST + s_cur));
      }
    }
  }
}

// ===================================================================================== host side
template <typename T>
static kldi_status up(T** dst, const std::vector<T>& v, cudaStream_t st) {
  KLDI_CUDA(cudaMalloc((void**)dst, std::max<size_t>(1, v.size()) * sizeof(T)));
  if (!v.empty()) KLDI_CUDA(cudaMemcpyAsync(*dst, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice, st));
  return KLDI_OK;
}

// Builds the pass/item tables for every panel size that occurs, the G_p workspace offsets and the
// issued-FLOP count of the V kernel (plan stage, once per geometry).
kldi_status vsched_upload(kldi_plan* P, const std::vector<int32_t>& h_kp, const std::vector<int32_t>& h_sh_ao0) {
  int max_nb = 0;
  for (int32_t k : h_kp) max_nb = std::max(max_nb, (k + 7) >> 3);
  std::vector<int64_t> count(max_nb + 1, 0);
  for (int32_t k : h_kp) count[(k + 7) >> 3]++;
  kldi_status rc;
  for (int m = 0; m < (P->want_grad ? 2 : 1); ++m) {
    std::vector<int32_t> ptr(max_nb + 2, 0);
    std::vector<VPass> passes;
    std::vector<VItem> items;
    double fexec = 0, fcrit = 0;
    for (int nb = 0; nb <= max_nb; ++nb) {
      ptr[nb] = (int32_t)passes.size();
      if (nb == 0 || count[nb] == 0) continue;
      vsched_build(nb, m == 1, passes, items);
      for (size_t i = ptr[nb]; i < passes.size(); ++i) {
        fexec += (double)count[nb] * passes[i].units * (2.0 * 8 * 8 * GB);  // units: 8x8 blocks
        fcrit += (double)count[nb] * passes[i].smsp_load * 4 * (2.0 * 8 * 8 * GB);  // 4 scheduler partitions
      }
    }
    ptr[max_nb + 1] = (int32_t)passes.size();
    if ((rc = up(&P->d_vsched_ptr[m], ptr, P->stream)) != KLDI_OK) return rc;
    VPass* dp = nullptr;
    VItem* di = nullptr;
    if ((rc = up(&dp, passes, P->stream)) != KLDI_OK) return rc;
    P->d_vpasses[m] = dp;
    if ((rc = up(&di, items, P->stream)) != KLDI_OK) return rc;
    P->d_vitems[m] = di;
    // workspace offsets of G_p: LDA strip-packed triangle, GGA square
    std::vector<int64_t> goff(h_kp.size() + 1, 0);
    for (size_t p = 0; p < h_kp.size(); ++p) {
      const int64_t k8 = (h_kp[p] + 7) & ~7, ns = (k8 + 15) / 16;
      goff[p + 1] = goff[p] + (m == 1 ? k8 * k8 : 16 * ns * k8 - 128 * ns * (ns - 1));
    }
    P->gram_elems[m] = goff.back();
    if ((rc = up(&P->d_gram_off[m], goff, P->stream)) != KLDI_OK) return rc;
    if (m == (P->want_grad ? 1 : 0)) {
      P->stats.flops_v_exec = fexec;
      P->stats.flops_v_crit = fcrit;
    }
  }
  std::vector<int32_t> ao_shell;
  for (size_t s = 0; s + 1 < h_sh_ao0.size(); ++s)
    for (int c = h_sh_ao0[s]; c < h_sh_ao0[s + 1]; ++c) ao_shell.push_back((int32_t)s);
  if ((rc = up(&P->d_ao_shell, ao_shell, P->stream)) != KLDI_OK) return rc;
  KLDI_CUDA(cudaStreamSynchronize(P->stream));  // the host vectors go out of scope
  return KLDI_OK;
}

// GGA: Z = 1/2 wv0 Phi + sum_c wv_c d_c Phi from the stored tiles, written in the V layout; HBM-bound.
__global__ void __launch_bounds__(128) k_build_z(const int32_t* __restrict__ kp, const int64_t* __restrict__ panel_off,
                                                 int64_t n_pad, const double* __restrict__ wv_s,
                                                 const double* __restrict__ phi, const double* __restrict__ d0,
                                                 const double* __restrict__ d1, const double* __restrict__ d2,
                                                 double* __restrict__ z) {
  const int p = blockIdx.x, t = threadIdx.x;
  const int64_t g = (int64_t)p * GB + t;
  const double w0 = 0.5 * wv_s[g], w1 = wv_s[n_pad + g], w2 = wv_s[2 * n_pad + g], w3 = wv_s[3 * n_pad + g];
  const int64_t o0 = panel_off[p] * GB + t;
  const int K = kp[p], K8 = (K + 7) & ~7;
  for (int k = 0; k < K; ++k) {
    const int64_t o = o0 + (int64_t)k * GB;
    z[vlayout_off(panel_off[p], K8, k, t)] = w0 * phi[o] + w1 * d0[o] + w2 * d1[o] + w3 * d2[o];
  }
}

// Fixed-point mode (EPI = 2): a bound on every partial sum of every V entry.  |G_p[i,j]| <= s_p a_pi a_pj with
// s_p = sum_{g in p} |wv_g| (GGA: 1/2|wv_0| + |wv_1| + |wv_2| + |wv_3|, the weights of Z) and a_pq the block maxima
// of the filter (Eq. 11), so by Cauchy-Schwarz |sum_p G_p[i,j]| <= sqrt(b_i b_j) <= max_q b_q,
// b_q = sum_{p in BCS(C) column q} s_p a_pq^2.  Fixed reduction trees and an associative max: the bound, and with it
// V, is reproducible.
__global__ void __launch_bounds__(256) k_fx_block_sums(int64_t n_blocks, int64_t n_pad, int ncomp,
                                                       const double* __restrict__ wv_s, double* __restrict__ s_p) {
  const int64_t p = (int64_t)blockIdx.x * 8 + (threadIdx.x >> 5);
  const int lane = threadIdx.x & 31;
  if (p >= n_blocks) return;
  double a = 0.0;
  for (int c = 0; c < ncomp; ++c) {
    double t = 0.0;
    for (int i = 0; i < 4; ++i) t += fabs(wv_s[c * n_pad + p * GB + lane + 32 * i]);
    a += (ncomp == 4 && c == 0) ? 0.5 * t : t;
  }
  for (int m = 16; m > 0; m >>= 1) a += __shfl_xor_sync(0xffffffffu, a, m);
  if (lane == 0) s_p[p] = a;
}
// one CTA per AO shell (a BCS(C) column can hold thousands of grid blocks)
__global__ void __launch_bounds__(256) k_fx_bound(const int32_t* __restrict__ col_ptr, const int32_t* __restrict__ row_idx,
                                                  const int32_t* __restrict__ pos, const double* __restrict__ amax,
                                                  const double* __restrict__ s_p, double* __restrict__ bound) {
  __shared__ double red[8];
  const int q = blockIdx.x, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  double b = 0.0;
  for (int e = col_ptr[q] + threadIdx.x; e < col_ptr[q + 1]; e += 256) {
    const double a = amax[pos[e]];
    b += s_p[row_idx[e]] * a * a;
  }
  for (int m = 16; m > 0; m >>= 1) b += __shfl_xor_sync(0xffffffffu, b, m);
  if (lane == 0) red[warp] = b;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < 8; ++w) b += red[w];
    // b >= 0: the bit pattern of a non-negative double orders like the value
    atomicMax(reinterpret_cast<unsigned long long*>(bound), (unsigned long long)__double_as_longlong(b));
  }
}

static kldi_status launch_fx_bound(kldi_plan* P, bool gga) {
  if (!P->d_fx) KLDI_CUDA(cudaMalloc(&P->d_fx, sizeof(double) * (size_t)(P->n_blocks + 1)));
  KLDI_CUDA(cudaMemsetAsync(P->d_fx, 0, sizeof(double), P->stream));
  k_fx_block_sums<<<(int)((P->n_blocks + 7) / 8), 256, 0, P->stream>>>(P->n_blocks, P->n_pad, gga ? 4 : 1, P->d_wv_s,
                                                                      P->d_fx + 1);
  KLDI_LAUNCHED(P);
  k_fx_bound<<<P->n_shells, 256, 0, P->stream>>>(P->d_col_ptr, P->d_row_idx, P->d_pos, P->d_blk_amax, P->d_fx + 1,
                                                 P->d_fx);
  KLDI_LAUNCHED(P);
  return KLDI_OK;
}

template <bool GGA, int EPI>
static kldi_status launch_vgram(kldi_plan* P, const double* phi_v = nullptr) {
  {
    const kldi_status rc_attr = ensure_smem_attr((const void*)k_vgram<GGA, EPI>, vg::SMEM_BYTES, P->device);
    if (rc_attr != KLDI_OK) return rc_attr;
  }
  const int m = GGA ? 1 : 0;
  const int grid = P->n_sm < P->n_tasks ? P->n_sm : P->n_tasks;
  k_vgram<GGA, EPI><<<grid, 32 * (V_WARPS + 1), vg::SMEM_BYTES, P->stream>>>(
      P->d_tasks, P->n_tasks, P->d_ticket, P->d_kp, P->d_panel_off, P->d_colidx, phi_v ? phi_v : P->d_phi_v, P->d_z,
      P->d_wv_s,
      P->d_vsched_ptr[m], static_cast<const VPass*>(P->d_vpasses[m]), static_cast<const VItem*>(P->d_vitems[m]),
      P->n_ao, P->d_Vp, P->d_gram_off[m], P->d_gram, P->d_fx);
  KLDI_LAUNCHED(P);
  return KLDI_OK;
}

// ===================================================================================== H5a fixed-order reduce
// Deterministic mode: V[i, :] = sum over the grid blocks p that retain AO i (BCS(C) column of its shell,
// ascending p: PAPER.md:466-470) of row r_p(i) of G_p, scattered through colidx.  One warp per plan AO row, the
// row accumulated in shared memory in that fixed order: no atomics, bitwise reproducible ("partial sums
// contributing to the same output tile are accumulated before the final write-back").
template <bool GGA>
__global__ void __launch_bounds__(128) k_vreduce(int n_ao, const int32_t* __restrict__ ao_shell,
                                                 const int32_t* __restrict__ sh_ao0, const int32_t* __restrict__ col_ptr,
                                                 const int32_t* __restrict__ row_idx, const int32_t* __restrict__ pos,
                                                 const int32_t* __restrict__ blk_col0, const int32_t* __restrict__ kp,
                                                 const int64_t* __restrict__ panel_off,
                                                 const int64_t* __restrict__ gram_off,
                                                 const int32_t* __restrict__ colidx, const double* __restrict__ G,
                                                 double* __restrict__ Vp) {
  extern __shared__ double rowbuf[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int i = blockIdx.x * (blockDim.x >> 5) + warp;
  if (i >= n_ao) return;
  double* buf = rowbuf + (size_t)warp * n_ao;
  for (int j = lane; j < n_ao; j += 32) buf[j] = 0.0;
  __syncwarp();
  const int q = ao_shell[i], a = i - sh_ao0[q];
  const int e_end = col_ptr[q + 1];
  for (int e0 = col_ptr[q]; e0 < e_end; e0 += 32) {
    // lane-parallel metadata of up to 32 contributions
    int64_t m_row = 0, m_base = 0;
    int m_c0 = 0, m_K = 0;
    if (e0 + lane < e_end) {
      const int p = row_idx[e0 + lane];
      const int r = blk_col0[pos[e0 + lane]] + a;
      m_K = kp[p];
      const int K8 = (m_K + 7) & ~7;
      m_base = panel_off[p];
      if (GGA) {
        m_row = gram_off[p] + (int64_t)r * K8;
        m_c0 = 0;
      } else {
        const int sx = r >> 4;
        m_row = gram_off[p] + (int64_t)16 * sx * K8 - (int64_t)128 * sx * (sx - 1) +
                (int64_t)(r - 16 * sx) * (K8 - 16 * sx) - 16 * sx;
        m_c0 = r;
      }
    }
    const int n = min(32, e_end - e0);
    // 4 contributions at a time: all their loads are issued before the first dependent shared-memory add, so
    // one memory latency is paid per group instead of per contribution; the adds stay in ascending-p order.
    constexpr int NU = 4, NCH = 3;
    for (int t0 = 0; t0 < n; t0 += NU) {
      int64_t row[NU], base[NU];
      int c0[NU], K[NU], jj[NU][NCH];
      double vv[NU][NCH];
#pragma unroll
      for (int u = 0; u < NU; ++u) {
        const int t = min(t0 + u, 31);
        row[u] = __shfl_sync(0xffffffffu, m_row, t);
        base[u] = __shfl_sync(0xffffffffu, m_base, t);
        c0[u] = __shfl_sync(0xffffffffu, m_c0, t);
        K[u] = (t0 + u < n) ? __shfl_sync(0xffffffffu, m_K, t) : 0;
#pragma unroll
        for (int ch = 0; ch < NCH; ++ch) {
          const int c = c0[u] + lane + 32 * ch;
          const bool ok = c < K[u];
          jj[u][ch] = ok ? __ldg(colidx + base[u] + c) : -1;
          vv[u][ch] = ok ? __ldcs(G + row[u] + c) : 0.0;
        }
      }
#pragma unroll
      for (int u = 0; u < NU; ++u) {
#pragma unroll
        for (int ch = 0; ch < NCH; ++ch)
          if (jj[u][ch] >= 0) buf[jj[u][ch]] += vv[u][ch];
        for (int c = c0[u] + lane + 32 * NCH; c < K[u]; c += 32) buf[colidx[base[u] + c]] += G[row[u] + c];
        __syncwarp();
      }
    }
  }
  for (int j = (GGA ? 0 : i) + lane; j < n_ao; j += 32) Vp[(int64_t)i * n_ao + j] = buf[j];
}

template <bool GGA>
static kldi_status launch_vreduce(kldi_plan* P) {
  const size_t row_bytes = sizeof(double) * (size_t)P->n_ao;
  int wpb = (int)std::min<size_t>(4, (220 * 1024) / row_bytes);
  if (wpb < 1) {
    set_error("deterministic V mode: n_ao = %d exceeds the shared-memory row buffer (28160)", P->n_ao);
    return KLDI_EINVAL;
  }
  const size_t smem = wpb * row_bytes;
  KLDI_CUDA(cudaFuncSetAttribute(k_vreduce<GGA>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const int m = GGA ? 1 : 0;
  k_vreduce<GGA><<<(P->n_ao + wpb - 1) / wpb, 32 * wpb, smem, P->stream>>>(
      P->n_ao, P->d_ao_shell, P->d_sh_ao0, P->d_col_ptr, P->d_row_idx, P->d_pos, P->d_blk_col0, P->d_kp,
      P->d_panel_off, P->d_gram_off[m], P->d_colidx, P->d_gram, P->d_Vp);
  KLDI_LAUNCHED(P);
  return KLDI_OK;
}

kldi_status launch_vxc(kldi_plan* P, bool gga) {
  KLDI_CUDA(cudaMemsetAsync(P->d_ticket, 0, sizeof(int32_t) * 4, P->stream));
  if (P->v_mode != 1) KLDI_CUDA(cudaMemsetAsync(P->d_Vp, 0, sizeof(double) * (size_t)P->n_ao * P->n_ao, P->stream));
  if (P->n_tasks == 0) {
    if (P->v_mode == 1) KLDI_CUDA(cudaMemsetAsync(P->d_Vp, 0, sizeof(double) * (size_t)P->n_ao * P->n_ao, P->stream));
    return KLDI_OK;
  }
  if (gga) {
    k_build_z<<<(int)P->n_blocks, 128, 0, P->stream>>>(P->d_kp, P->d_panel_off, P->n_pad, P->d_wv_s, P->d_phi,
                                                       P->d_dphi[0], P->d_dphi[1], P->d_dphi[2], P->d_z);
    KLDI_LAUNCHED(P);
  }
  if (P->v_mode == 0) return gga ? launch_vgram<true, 0>(P) : launch_vgram<false, 0>(P);
  if (P->v_mode == 2) {
    kldi_status rc = launch_fx_bound(P, gga);
    if (rc != KLDI_OK) return rc;
    return gga ? launch_vgram<true, 2>(P) : launch_vgram<false, 2>(P);
  }
  // deterministic mode: G_p partials to the workspace, then the fixed-order reduce
  const int m = gga ? 1 : 0;
  if (P->gram_cap < P->gram_elems[m]) {
    if (P->d_gram) KLDI_CUDA(cudaFree(P->d_gram));
    P->d_gram = nullptr;
    P->gram_cap = 0;
    KLDI_CUDA(cudaMalloc(&P->d_gram, sizeof(double) * (size_t)std::max<int64_t>(1, P->gram_elems[m])));
    P->gram_cap = P->gram_elems[m];
  }
  kldi_status rc = gga ? launch_vgram<true, 1>(P) : launch_vgram<false, 1>(P);
  if (rc != KLDI_OK) return rc;
  return gga ? launch_vreduce<true>(P) : launch_vreduce<false>(P);
}

// rho layout ([column][128 rows]) -> V layout (vlayout_off) of one store; HBM-bound.
__global__ void __launch_bounds__(128) k_relayout_v(const int64_t* __restrict__ panel_off,
                                                    const double* __restrict__ src, double* __restrict__ dst) {
  const int p = blockIdx.x, t = threadIdx.x;
  const int64_t base = panel_off[p];
  const int K8 = (int)(panel_off[p + 1] - base);
  for (int k = 0; k < K8; ++k) dst[vlayout_off(base, K8, k, t)] = src[(base + k) * GB + t];
}

// V^tau = 1/2 sum_c (d_c Phi)^T diag(wv) (d_c Phi): three LDA-form Gram builds that accumulate
// into the same plan-order V; wv_s already carries the 1/2.  The gradient stores are copied into the V layout ONCE, at
// the first call (the geometry of a plan is fixed), not per call.  Mode 1 (workspace + reduce) does not accumulate across
// launches, so it runs as mode 2 here, which is reproducible and free of FP64 atomics as well.
kldi_status launch_vtau(kldi_plan* P) {
  KLDI_CUDA(cudaMemsetAsync(P->d_Vp, 0, sizeof(double) * (size_t)P->n_ao * P->n_ao, P->stream));
  if (P->n_tasks == 0) return KLDI_OK;
  kldi_status rc;
  if (!P->d_dphi_v[0]) {
    const size_t tile_bytes = sizeof(double) * GB * (size_t)(P->total_cols + 64);
    for (int c = 0; c < 3; ++c) {
      KLDI_CUDA(cudaMalloc(&P->d_dphi_v[c], tile_bytes));
      KLDI_CUDA(cudaMemsetAsync(P->d_dphi_v[c], 0, tile_bytes, P->stream));
      k_relayout_v<<<(int)P->n_blocks, 128, 0, P->stream>>>(P->d_panel_off, P->d_dphi[c], P->d_dphi_v[c]);
      KLDI_LAUNCHED(P);
    }
    P->stats.phi_bytes += 3 * (int64_t)tile_bytes;
  }
  if (P->v_mode != 0 && (rc = launch_fx_bound(P, false)) != KLDI_OK) return rc;
  for (int c = 0; c < 3; ++c) {
    KLDI_CUDA(cudaMemsetAsync(P->d_ticket, 0, sizeof(int32_t) * 4, P->stream));
    rc = P->v_mode != 0 ? launch_vgram<false, 2>(P, P->d_dphi_v[c]) : launch_vgram<false, 0>(P, P->d_dphi_v[c]);
    if (rc != KLDI_OK) return rc;
  }
  return KLDI_OK;
}

}  // namespace kldi

extern "C" {

kldi_status kldi_vsched_export(int nb, int square, int32_t* passes, int32_t* items, int64_t cap, int64_t* n_passes) {
  if (nb < 0 || nb > 4095 || !n_passes) {
    kldi::set_error("kldi_vsched_export: bad argument");
    return KLDI_EINVAL;
  }
  std::vector<kldi::VPass> P;
  std::vector<kldi::VItem> I;
  if (nb > 0) kldi::vsched_build(nb, square != 0, P, I);
  *n_passes = (int64_t)P.size();
  if (!passes || !items || cap < *n_passes) return KLDI_OK;
  static_assert(sizeof(kldi::VPass) == 32 && sizeof(kldi::VItem) == 8, "export layout");
  static_assert(kldi::V_ITEMS <= 32, "kldi_vsched_export documents 32 item slots per pass");
  memset(items, 0, (size_t)*n_passes * 32 * sizeof(kldi::VItem));
  for (size_t i = 0; i < P.size(); ++i) {
    kldi::VPass q = P[i];
    q.pad1 = kldi::V_WARPS | (kldi::V_SLOTS << 8);  // shape of the schedule, for the caller
    memcpy(passes + 8 * i, &q, sizeof(q));
    memcpy(items + 64 * i, I.data() + i * kldi::V_ITEMS, kldi::V_ITEMS * sizeof(kldi::VItem));
  }
  return KLDI_OK;
}

int64_t kldi_vlayout_offset(int64_t panel_off, int32_t K8, int32_t col, int32_t row) {
  return kldi::vlayout_off(panel_off, K8, col, row);
}

}  // extern "C"
