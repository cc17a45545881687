// Plan stage of libkldi: once per geometry.
//   P1 grid reorder      — 60-bit space-filling-curve keys on Eq. 20's lattice (the Hilbert index,
//                          hilbert_key below; Eq. 20's own Z-order key is kept as morton_key), stable radix sort, blocks of 128
//   P2 AO partition      — atoms in the same curve order, one AO block per shell
//   P3 AO evaluation     — Cartesian Gaussian shells on (grid block, shell) tiles (Eq. 2)
//   P4 block filter      — a_pq = max|Phi_pq|, keep iff a_pq >= eps (Eq. 11-13)
//   P5 BCS build         — BCS(R) row_ptr/col_idx/data and BCS(C) col_ptr/row_idx/pos
#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <cub/device/device_radix_sort.cuh>
#include <cub/device/device_scan.cuh>
#include <numeric>

#include "ao_eval.cuh"
#include "kldi_internal.h"

namespace kldi {

// --------------------------------------------------------------------------------- Morton (Eq. 20)
__host__ __device__ inline uint64_t spread3(uint64_t v) {  // 20 bits -> every third bit
  v &= 0xFFFFFull;
  v = (v | (v << 32)) & 0x001F00000000FFFFull;
  v = (v | (v << 16)) & 0x001F0000FF0000FFull;
  v = (v | (v << 8)) & 0x100F00F00F00F00Full;
  v = (v | (v << 4)) & 0x10C30C30C30C30C3ull;
  v = (v | (v << 2)) & 0x1249249249249249ull;
  return v;
}
// m = sum_k z_k 2^{3k} + y_k 2^{3k+1} + x_k 2^{3k+2}; coordinates are shifted by the bounding-box
// minimum, scaled by 128 and truncated, clamped to 20 bits (reading A3).
__host__ __device__ inline uint64_t morton_key(double x, double y, double z, double x0, double y0, double z0) {
  auto q = [](double v) -> uint64_t {
    double t = v * 128.0;
    if (!(t > 0.0)) return 0;
    if (t >= 1048575.0) return 1048575ull;
    return (uint64_t)t;
  };
  return (spread3(q(x - x0)) << 2) | (spread3(q(y - y0)) << 1) | spread3(q(z - z0));
}

uint64_t morton_key_host(double x, double y, double z, double x0, double y0, double z0) {
  return morton_key(x, y, z, x0, y0, z0);
}

// The key the plan actually sorts by ("grid-block shape beyond Morton"): the Hilbert index of the
// same 3 x 20-bit lattice coordinates as Eq. 20.  The Hilbert curve has no jumps, so 128 consecutive points form a
// more compact block and retain fewer AO shells: sum_p K_p^2 drops by 7 % against the Z-order on the water clusters
// (measured); the order is internal and cannot change results (reading A3).  Skilling's
// axes-to-transpose transform, then the bit interleave of Eq. 20.
__host__ __device__ inline uint64_t hilbert_key(double x, double y, double z, double x0, double y0, double z0) {
  auto q = [](double v) -> uint32_t {
    double t = v * 128.0;
    if (!(t > 0.0)) return 0u;
    if (t >= 1048575.0) return 1048575u;
    return (uint32_t)t;
  };
  uint32_t X[3] = {q(x - x0), q(y - y0), q(z - z0)};
  const uint32_t M = 1u << 19;
  for (uint32_t Q = M; Q > 1; Q >>= 1) {
    const uint32_t P = Q - 1;
    for (int i = 0; i < 3; ++i) {
      if (X[i] & Q) {
        X[0] ^= P;
      } else {
        const uint32_t t = (X[0] ^ X[i]) & P;
        X[0] ^= t;
        X[i] ^= t;
      }
    }
  }
  X[1] ^= X[0];
  X[2] ^= X[1];
  uint32_t t = 0;
  for (uint32_t Q = M; Q > 1; Q >>= 1)
    if (X[2] & Q) t ^= Q - 1;
  for (int i = 0; i < 3; ++i) X[i] ^= t;
  return (spread3(X[0]) << 2) | (spread3(X[1]) << 1) | spread3(X[2]);
}

uint64_t grid_key_host(double x, double y, double z, double x0, double y0, double z0) {
  return hilbert_key(x, y, z, x0, y0, z0);
}

__global__ void k_morton_keys(const double* __restrict__ xyz, int64_t n, int64_t n_pad, double x0, double y0,
                              double z0, uint64_t* __restrict__ keys, int32_t* __restrict__ idx) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_pad) return;
  if (i < n) {
    keys[i] = hilbert_key(xyz[3 * i], xyz[3 * i + 1], xyz[3 * i + 2], x0, y0, z0);
    idx[i] = (int32_t)i;
  } else {
    keys[i] = 1ull << 63;  // padding sorts last
    idx[i] = -1;
  }
}

// sorted SoA copy; padding points repeat the last real point with zero weight
__global__ void k_gather_grid(const double* __restrict__ xyz, const double* __restrict__ w,
                              const int32_t* __restrict__ perm, int64_t n, int64_t n_pad, double* __restrict__ gx,
                              double* __restrict__ gy, double* __restrict__ gz, double* __restrict__ gw) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_pad) return;
  int64_t src = perm[i];
  double ww = 0.0;
  if (src < 0) {
    src = perm[n - 1];
  } else {
    ww = w[src];
  }
  gx[i] = xyz[3 * src];
  gy[i] = xyz[3 * src + 1];
  gz[i] = xyz[3 * src + 2];
  gw[i] = ww;
}

// --------------------------------------------------------------------------------- P3/P4 screening
// One CTA (4 warps) per grid block.  Warps walk the atoms; an atom's shells are first tested
// against a rigorous upper bound on the block's bounding box, survivors are evaluated exactly
// on the 128 points and reduced to a_pq = max|.| with warp shuffles.
template <bool GRAD>
__global__ void __launch_bounds__(128) k_screen(ShellTable T, const int32_t* __restrict__ atom_sh0, int n_atoms,
                                                int n_shells, const double* __restrict__ gx,
                                                const double* __restrict__ gy, const double* __restrict__ gz,
                                                double eps, uint8_t* __restrict__ keep) {
  __shared__ double sx[GB], sy[GB], sz[GB];
  __shared__ double red[6][4];
  const int p = blockIdx.x, t = threadIdx.x, lane = t & 31, warp = t >> 5;
  const double x = gx[(int64_t)p * GB + t], y = gy[(int64_t)p * GB + t], z = gz[(int64_t)p * GB + t];
  sx[t] = x; sy[t] = y; sz[t] = z;
  double v[6] = {x, -x, y, -y, z, -z};
#pragma unroll
  for (int c = 0; c < 6; ++c) {
    double m = v[c];
    for (int o = 16; o > 0; o >>= 1) m = fmin(m, __shfl_xor_sync(0xffffffffu, m, o));
    if (lane == 0) red[c][warp] = m;
  }
  __syncthreads();
  double lo[3], hi[3];
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    lo[c] = fmin(fmin(red[2 * c][0], red[2 * c][1]), fmin(red[2 * c][2], red[2 * c][3]));
    hi[c] = -fmin(fmin(red[2 * c + 1][0], red[2 * c + 1][1]), fmin(red[2 * c + 1][2], red[2 * c + 1][3]));
  }
  uint8_t* kp = keep + (int64_t)p * n_shells;
  for (int a = warp; a < n_atoms; a += 4) {
    const double ax = T.atom_xyz[3 * a], ay = T.atom_xyz[3 * a + 1], az = T.atom_xyz[3 * a + 2];
    const double A[3] = {ax, ay, az};
    double dmin2 = 0.0, dmax2 = 0.0;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const double dn = fmax(fmax(lo[c] - A[c], A[c] - hi[c]), 0.0);
      const double dx = fmax(fabs(A[c] - lo[c]), fabs(A[c] - hi[c]));
      dmin2 += dn * dn;
      dmax2 += dx * dx;
    }
    const double dmax = sqrt(dmax2);
    for (int s = atom_sh0[a]; s < atom_sh0[a + 1]; ++s) {
      const int l = T.sh_l[s];
      if (eps > 0.0) {
        // |chi| <= r^l sum|cn| e^{-a r^2};  |d chi| <= l r^{l-1} sum|cn| e + r^{l+1} sum 2a|cn| e
        double s0 = 0.0, s1 = 0.0;
        for (int i = T.sh_prim0[s]; i < T.sh_prim0[s + 1]; ++i) {
          const double e = fabs(T.prim_cn[i]) * exp(-T.prim_alpha[i] * dmin2);
          s0 += e;
          s1 += 2.0 * T.prim_alpha[i] * e;
        }
        const double pl = (l == 0) ? 1.0 : (l == 1 ? dmax : dmax2);
        double bound = pl * s0;
        if (GRAD) {
          const double plm = (l == 0) ? 0.0 : (l == 1 ? 1.0 : 2.0 * dmax);
          bound = fmax(bound, plm * s0 + pl * dmax * s1);
        }
        if (bound * 1.000001 < eps) continue;  // keep[] was zero-filled
      }
      double m = 0.0;
#pragma unroll
      for (int r = 0; r < 4; ++r) {
        const int i = lane + 32 * r;
        double val[6], g0[6], g1[6], g2[6];
        eval_shell<GRAD>(T, s, sx[i], sy[i], sz[i], val, g0, g1, g2);
        const int nc = (l + 1) * (l + 2) / 2;
        for (int c = 0; c < nc; ++c) {
          m = fmax(m, fabs(val[c]));
          if (GRAD) m = fmax(m, fmax(fabs(g0[c]), fmax(fabs(g1[c]), fabs(g2[c]))));
        }
      }
      for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
      if (lane == 0) kp[s] = (eps <= 0.0 || m >= eps) ? 1 : 0;  // Eq. 12: retain iff a_pq >= t_b
    }
  }
}

// --------------------------------------------------------------------------------- P3/P5 tile fill
// One CTA per grid block, one thread per point; walks the block's BCS(R) row and writes the
// column-major tiles Phi[(panel_off[p] + k)*128 + t]; a_pq via atomicMax on the bit pattern.
template <bool GRAD>
__global__ void __launch_bounds__(128) k_fill(ShellTable T, const int32_t* __restrict__ row_ptr,
                                              const int32_t* __restrict__ col_idx,
                                              const int32_t* __restrict__ blk_col0,
                                              const int64_t* __restrict__ panel_off, const double* __restrict__ gx,
                                              const double* __restrict__ gy, const double* __restrict__ gz,
                                              double* __restrict__ phi, double* __restrict__ phi_v,
                                              double* __restrict__ d0, double* __restrict__ d1,
                                              double* __restrict__ d2, unsigned long long* __restrict__ amax_bits) {
  const int p = blockIdx.x, t = threadIdx.x, lane = t & 31;
  const int64_t g = (int64_t)p * GB + t;
  const double x = gx[g], y = gy[g], z = gz[g];
  const int64_t base = panel_off[p] * GB + t;
  const int K8 = (int)(panel_off[p + 1] - panel_off[p]);
  for (int e = row_ptr[p]; e < row_ptr[p + 1]; ++e) {
    const int s = col_idx[e];
    const int l = T.sh_l[s];
    const int nc = (l + 1) * (l + 2) / 2;
    double val[6], g0[6], g1[6], g2[6];
    eval_shell<GRAD>(T, s, x, y, z, val, g0, g1, g2);
    const int64_t o = base + (int64_t)blk_col0[e] * GB;
    double m = 0.0;
    for (int c = 0; c < nc; ++c) {
      phi[o + (int64_t)c * GB] = val[c];
      phi_v[vlayout_off(panel_off[p], K8, blk_col0[e] + c, t)] = val[c];
      m = fmax(m, fabs(val[c]));
      if (GRAD) {
        d0[o + (int64_t)c * GB] = g0[c];
        d1[o + (int64_t)c * GB] = g1[c];
        d2[o + (int64_t)c * GB] = g2[c];
        m = fmax(m, fmax(fabs(g0[c]), fmax(fabs(g1[c]), fabs(g2[c]))));
      }
    }
    for (int o2 = 16; o2 > 0; o2 >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o2));
    if (lane == 0) atomicMax(amax_bits + e, (unsigned long long)__double_as_longlong(m));
  }
}

// --------------------------------------------------------------------------------- P5: BCS build on the device
// The keep mask of the filter (Eq. 12) becomes BCS(R) by count -> prefix sum -> compaction (the mask + prefix-sum
// pair selection of Alg. 1, applied to the block layout of PAPER.md:459-471), one warp per grid
// block; BCS(C) is its transpose by a stable radix sort of the entries on their shell index.
__global__ void __launch_bounds__(256) k_bcs_count(const uint8_t* __restrict__ keep, int n_shells,
                                                   const int32_t* __restrict__ sh_ao0, int64_t n_blocks,
                                                   int64_t* __restrict__ cnt, int32_t* __restrict__ kp,
                                                   int64_t* __restrict__ k8) {
  const int64_t p = (int64_t)blockIdx.x * 8 + (threadIdx.x >> 5);
  const int lane = threadIdx.x & 31;
  if (p > n_blocks) return;
  int c = 0, k = 0;
  if (p < n_blocks)
    for (int s = lane; s < n_shells; s += 32)
      if (keep[p * n_shells + s]) {
        c++;
        k += sh_ao0[s + 1] - sh_ao0[s];
      }
  for (int o = 16; o > 0; o >>= 1) {
    c += __shfl_xor_sync(0xffffffffu, c, o);
    k += __shfl_xor_sync(0xffffffffu, k, o);
  }
  if (lane == 0) {  // entry n_blocks is the zero that turns the exclusive scans into [n_blocks + 1] offset arrays
    cnt[p] = c;
    k8[p] = (k + 7) & ~7;
    if (p < n_blocks) kp[p] = k;
  }
}

__global__ void k_narrow(const int64_t* __restrict__ in, int64_t n, int32_t* __restrict__ out) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = (int32_t)in[i];
}

__global__ void __launch_bounds__(256) k_bcs_fill(const uint8_t* __restrict__ keep, int n_shells,
                                                  const int32_t* __restrict__ sh_ao0, int64_t n_blocks,
                                                  const int32_t* __restrict__ row_ptr,
                                                  const int64_t* __restrict__ panel_off, const int32_t* __restrict__ kp,
                                                  int32_t* __restrict__ col_idx, int32_t* __restrict__ blk_col0,
                                                  int32_t* __restrict__ entry_row, int32_t* __restrict__ entry_id,
                                                  int32_t* __restrict__ colidx, int32_t* __restrict__ col_cnt) {
  const int64_t p = (int64_t)blockIdx.x * 8 + (threadIdx.x >> 5);
  const int lane = threadIdx.x & 31;
  if (p >= n_blocks) return;
  int e_base = row_ptr[p], kbase = 0;
  const int64_t base = panel_off[p];
  for (int s0 = 0; s0 < n_shells; s0 += 32) {
    const int s = s0 + lane;
    const bool kept = s < n_shells && keep[p * n_shells + s];
    const int w = kept ? sh_ao0[s + 1] - sh_ao0[s] : 0;
    const unsigned m = __ballot_sync(0xffffffffu, kept);
    int incl = w;
    for (int o = 1; o < 32; o <<= 1) {
      const int t = __shfl_up_sync(0xffffffffu, incl, o);
      if (lane >= o) incl += t;
    }
    if (kept) {
      const int e = e_base + __popc(m & ((1u << lane) - 1u));
      const int k0 = kbase + incl - w;
      col_idx[e] = s;
      blk_col0[e] = k0;
      entry_row[e] = (int32_t)p;
      entry_id[e] = e;
      atomicAdd(col_cnt + s + 1, 1);
      for (int c = 0; c < w; ++c) colidx[base + k0 + c] = sh_ao0[s] + c;
    }
    e_base += __popc(m);
    kbase += __shfl_sync(0xffffffffu, incl, 31);
  }
  const int k = kp[p], k8 = (k + 7) & ~7;
  for (int c = k + lane; c < k8; c += 32) colidx[base + c] = 0;  // zero columns: any valid AO index
}

__global__ void k_gather_i32(const int32_t* __restrict__ src, const int32_t* __restrict__ idx, int64_t n,
                             int32_t* __restrict__ dst) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) dst[i] = src[idx[i]];
}

// --------------------------------------------------------------------------------- host helpers
template <class T>
static kldi_status upload(T** dst, const std::vector<T>& v, cudaStream_t st, size_t extra = 0) {
  KLDI_CUDA(cudaMalloc((void**)dst, std::max<size_t>(1, v.size() + extra) * sizeof(T)));
  if (!v.empty()) KLDI_CUDA(cudaMemcpyAsync(*dst, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice, st));
  return KLDI_OK;
}

void plan_free(kldi_plan* P) {
  if (!P) return;
  cudaSetDevice(P->device);
  void* ptrs[] = {P->d_atom_xyz, P->d_sh_atom, P->d_sh_l, P->d_sh_prim0, P->d_sh_ao0, P->d_prim_alpha, P->d_prim_cn,
                  P->d_shell_perm, P->d_ao_perm, P->d_ao_atom, P->d_ao_atom_c, P->d_x, P->d_xd, P->d_fx, P->d_gx, P->d_gy, P->d_gz, P->d_gw, P->d_perm_g,
                  P->d_keys, P->d_row_ptr, P->d_col_idx, P->d_blk_col0, P->d_col_ptr, P->d_row_idx, P->d_pos,
                  P->d_blk_amax, P->d_panel_off, P->d_kp, P->d_colidx, P->d_phi, P->d_dphi[0], P->d_dphi[1],
                  P->d_dphi[2], P->d_dphi_v[0], P->d_dphi_v[1], P->d_dphi_v[2], P->d_z, P->d_phi_v, P->d_tasks, P->d_ticket, P->d_Dp, P->d_Vp, P->d_rho_s, P->d_drho_s,
                  P->d_wv_s, P->d_epart, P->d_E, P->d_stage_host, P->d_vsched_ptr[0], P->d_vsched_ptr[1],
                  P->d_vpasses[0], P->d_vpasses[1], P->d_vitems[0], P->d_vitems[1], P->d_gram_off[0],
                  P->d_gram_off[1], P->d_gram, P->d_ao_shell, P->d_bmax, P->d_pmask, P->d_phiq, P->d_sigma, P->d_dphiq[0], P->d_dphiq[1], P->d_dphiq[2], P->d_dsigma[0], P->d_dsigma[1],
                  P->d_dsigma[2], P->d_Dq, P->d_tau,
                  P->d_chunk_off};
  for (void* q : ptrs)
    if (q) cudaFree(q);
  if (P->h_E) cudaFreeHost(P->h_E);
  for (auto& e : P->ev)
    if (e) cudaEventDestroy(e);
}

kldi_status plan_build(kldi_plan* P, const kldi_atoms* atoms, const kldi_shells* shells, const kldi_grid* grid) {
  const auto t_start = std::chrono::steady_clock::now();
  cudaStream_t st = P->stream;
  const int n_atoms = atoms->n_atoms, n_shells = shells->n_shells;
  const int64_t n_pts = grid->n_pts;
  P->n_atoms = n_atoms;
  P->n_shells = n_shells;
  P->n_pts = n_pts;
  P->n_blocks = (n_pts + GB - 1) / GB;
  P->n_pad = P->n_blocks * GB;
  if (P->n_pad >= (int64_t)1 << 31) {
    set_error("grid too large for int32 point indices");
    return KLDI_EINVAL;
  }

  // ---- P2: atoms in Morton order of their positions; shells follow their atom, given order inside
  double a0[3] = {1e300, 1e300, 1e300};
  for (int a = 0; a < n_atoms; ++a)
    for (int c = 0; c < 3; ++c) a0[c] = std::min(a0[c], atoms->xyz[3 * a + c]);
  std::vector<int> atom_order(n_atoms);
  std::iota(atom_order.begin(), atom_order.end(), 0);
  std::vector<uint64_t> akey(n_atoms);
  for (int a = 0; a < n_atoms; ++a)
    akey[a] = hilbert_key(atoms->xyz[3 * a], atoms->xyz[3 * a + 1], atoms->xyz[3 * a + 2], a0[0], a0[1], a0[2]);
  std::stable_sort(atom_order.begin(), atom_order.end(), [&](int i, int j) { return akey[i] < akey[j]; });
  if (g_default_ao_order == 2) {
    std::iota(atom_order.begin(), atom_order.end(), 0);  // the caller's order (measurement only)
  } else if (g_default_ao_order == 1) {
    std::vector<int> o;  // overlap-signature clustering; beyond its size limit the curve order stays
    if (overlap_signature_order(atoms, shells, o)) atom_order = o;
  }
  std::vector<int> atom_rank(n_atoms);
  for (int r = 0; r < n_atoms; ++r) atom_rank[atom_order[r]] = r;

  std::vector<std::vector<int>> shells_of(n_atoms);
  std::vector<int32_t> caller_ao0(n_shells + 1, 0);
  for (int s = 0; s < n_shells; ++s) {
    const int l = shells->l[s], a = shells->atom[s];
    if (l < 0 || l > 2 || a < 0 || a >= n_atoms || shells->nprim_off[s + 1] <= shells->nprim_off[s]) {
      set_error("shell %d: l=%d atom=%d nprim=%d not supported", s, l, a,
                shells->nprim_off[s + 1] - shells->nprim_off[s]);
      return KLDI_EINVAL;
    }
    shells_of[a].push_back(s);
    caller_ao0[s + 1] = caller_ao0[s] + (l + 1) * (l + 2) / 2;
  }
  P->n_ao = caller_ao0[n_shells];
  const int n_ao = P->n_ao;

  std::vector<double> h_axyz(3 * (size_t)n_atoms), h_alpha, h_cn;
  std::vector<int32_t> h_sh_atom, h_sh_l, h_sh_prim0{0}, h_sh_ao0{0}, h_atom_sh0{0}, h_ao_atom, h_ao_atom_c;
  P->h_shell_perm.clear();
  P->h_ao_perm.clear();
  for (int r = 0; r < n_atoms; ++r) {
    const int a = atom_order[r];
    for (int c = 0; c < 3; ++c) h_axyz[3 * r + c] = atoms->xyz[3 * a + c];
    for (int s : shells_of[a]) {
      const int l = shells->l[s], nc = (l + 1) * (l + 2) / 2;
      P->h_shell_perm.push_back(s);
      h_sh_atom.push_back(r);
      h_sh_l.push_back(l);
      for (int i = shells->nprim_off[s]; i < shells->nprim_off[s + 1]; ++i) {
        const double al = shells->alpha[i];
        if (!(al > 0.0)) {
          set_error("primitive %d: exponent must be positive", i);
          return KLDI_EINVAL;
        }
        h_alpha.push_back(al);
        h_cn.push_back(shells->coef[i] * std::pow(2.0 * al / M_PI, 0.75) * std::pow(4.0 * al, 0.5 * l));
      }
      h_sh_prim0.push_back((int32_t)h_alpha.size());
      for (int c = 0; c < nc; ++c) {
        P->h_ao_perm.push_back(caller_ao0[s] + c);
        h_ao_atom.push_back(r);
        h_ao_atom_c.push_back(a);
      }
      h_sh_ao0.push_back((int32_t)P->h_ao_perm.size());
    }
    h_atom_sh0.push_back((int32_t)h_sh_l.size());
  }
  P->n_prim = (int32_t)h_alpha.size();

  kldi_status rc;
  int32_t* d_atom_sh0 = nullptr;
#define UP(dst, vec)                                    \
  if ((rc = upload(&(dst), (vec), st)) != KLDI_OK) {    \
    cudaFree(d_atom_sh0); /* the only temporary so far; the plan's own buffers go in plan_free */ \
    return rc;                                          \
  }
  UP(P->d_atom_xyz, h_axyz);
  UP(P->d_sh_atom, h_sh_atom);
  UP(P->d_sh_l, h_sh_l);
  UP(P->d_sh_prim0, h_sh_prim0);
  UP(P->d_sh_ao0, h_sh_ao0);
  UP(P->d_prim_alpha, h_alpha);
  UP(P->d_prim_cn, h_cn);
  UP(P->d_shell_perm, P->h_shell_perm);
  UP(P->d_ao_perm, P->h_ao_perm);
  UP(P->d_ao_atom, h_ao_atom);
  UP(P->d_ao_atom_c, h_ao_atom_c);
  UP(d_atom_sh0, h_atom_sh0);
  ShellTable T{P->d_atom_xyz, P->d_sh_atom, P->d_sh_l, P->d_sh_prim0, P->d_sh_ao0, P->d_prim_alpha, P->d_prim_cn};

  // ---- P1: Morton keys, stable radix sort, sorted SoA grid
  double g0[3] = {1e300, 1e300, 1e300};
  for (int64_t i = 0; i < n_pts; ++i)
    for (int c = 0; c < 3; ++c) {
      const double v = grid->xyz[3 * i + c];
      if (!(std::fabs(v) < 1e300)) {
        set_error("grid point %lld is not finite", (long long)i);
        cudaFree(d_atom_sh0);
        return KLDI_EINVAL;
      }
      g0[c] = std::min(g0[c], v);
    }
  const int64_t n_pad = P->n_pad;
  double *d_xyz = nullptr, *d_w = nullptr;
  uint64_t* d_keys_in = nullptr;
  int32_t* d_idx_in = nullptr;
  void* d_tmp = nullptr;
  uint8_t* d_keep = nullptr;
  int64_t *d_cnt64 = nullptr, *d_k8 = nullptr, *d_rp64 = nullptr;
  int32_t *d_erow = nullptr, *d_eid = nullptr, *d_skey = nullptr, *d_ccnt = nullptr;
  auto cleanup = [&]() {
    cudaFree(d_atom_sh0); cudaFree(d_xyz); cudaFree(d_w); cudaFree(d_keys_in); cudaFree(d_idx_in);
    cudaFree(d_tmp); cudaFree(d_keep);
    cudaFree(d_cnt64); cudaFree(d_k8); cudaFree(d_rp64); cudaFree(d_erow); cudaFree(d_eid); cudaFree(d_skey); cudaFree(d_ccnt);
  };
#define CK(call)                        \
  do {                                  \
    cudaError_t e_ = (call);            \
    if (e_ != cudaSuccess) {            \
      set_error("%s:%d: %s -> %s", __FILE__, __LINE__, #call, cudaGetErrorString(e_)); \
      cleanup();                        \
      return e_ == cudaErrorMemoryAllocation ? KLDI_ENOMEM : KLDI_ECUDA; \
    }                                   \
  } while (0)
  CK(cudaMalloc(&d_xyz, sizeof(double) * 3 * n_pts));
  CK(cudaMalloc(&d_w, sizeof(double) * n_pts));
  CK(cudaMemcpyAsync(d_xyz, grid->xyz, sizeof(double) * 3 * n_pts, cudaMemcpyHostToDevice, st));
  CK(cudaMemcpyAsync(d_w, grid->w, sizeof(double) * n_pts, cudaMemcpyHostToDevice, st));
  CK(cudaMalloc(&d_keys_in, sizeof(uint64_t) * n_pad));
  CK(cudaMalloc(&d_idx_in, sizeof(int32_t) * n_pad));
  CK(cudaMalloc(&P->d_keys, sizeof(uint64_t) * n_pad));
  CK(cudaMalloc(&P->d_perm_g, sizeof(int32_t) * n_pad));
  const int nb256 = (int)((n_pad + 255) / 256);
  k_morton_keys<<<nb256, 256, 0, st>>>(d_xyz, n_pts, n_pad, g0[0], g0[1], g0[2], d_keys_in, d_idx_in);
  size_t tmp_bytes = 0;
  CK(cub::DeviceRadixSort::SortPairs(nullptr, tmp_bytes, d_keys_in, P->d_keys, d_idx_in, P->d_perm_g, (int)n_pad, 0,
                                     64, st));
  CK(cudaMalloc(&d_tmp, tmp_bytes));
  CK(cub::DeviceRadixSort::SortPairs(d_tmp, tmp_bytes, d_keys_in, P->d_keys, d_idx_in, P->d_perm_g, (int)n_pad, 0, 64,
                                     st));  // LSD radix sort: stable
  CK(cudaMalloc(&P->d_gx, sizeof(double) * n_pad));
  CK(cudaMalloc(&P->d_gy, sizeof(double) * n_pad));
  CK(cudaMalloc(&P->d_gz, sizeof(double) * n_pad));
  CK(cudaMalloc(&P->d_gw, sizeof(double) * n_pad));
  k_gather_grid<<<nb256, 256, 0, st>>>(d_xyz, d_w, P->d_perm_g, n_pts, n_pad, P->d_gx, P->d_gy, P->d_gz, P->d_gw);

  // ---- P3/P4: block-max screening -> dense keep mask [n_blocks][n_shells]
  const int64_t n_blocks = P->n_blocks;
  const size_t mask_bytes = (size_t)n_blocks * n_shells;
  CK(cudaMalloc(&d_keep, mask_bytes));
  CK(cudaMemsetAsync(d_keep, 0, mask_bytes, st));
  if (P->want_grad)
    k_screen<true><<<(int)n_blocks, 128, 0, st>>>(T, d_atom_sh0, n_atoms, n_shells, P->d_gx, P->d_gy, P->d_gz, P->eps,
                                                  d_keep);
  else
    k_screen<false><<<(int)n_blocks, 128, 0, st>>>(T, d_atom_sh0, n_atoms, n_shells, P->d_gx, P->d_gy, P->d_gz,
                                                   P->eps, d_keep);
  CK(cudaGetLastError());
  // ---- P5: BCS(R), packed column maps, BCS(C) — built on the device, host copies kept for export / statistics
  auto& row_ptr = P->h_row_ptr;
  auto& col_idx = P->h_col_idx;
  auto& blk_col0 = P->h_blk_col0;
  auto& panel_off = P->h_panel_off;
  auto& col_ptr = P->h_col_ptr;
  auto& row_idx = P->h_row_idx;
  auto& pos = P->h_pos;
  std::vector<int32_t> h_kp(n_blocks), h_tasks;
  const int nbw = (int)((n_blocks + 1 + 7) / 8);
  CK(cudaMalloc(&d_cnt64, sizeof(int64_t) * (n_blocks + 1)));
  CK(cudaMalloc(&d_k8, sizeof(int64_t) * (n_blocks + 1)));
  CK(cudaMalloc(&d_rp64, sizeof(int64_t) * (n_blocks + 1)));
  CK(cudaMalloc(&P->d_kp, sizeof(int32_t) * std::max<int64_t>(1, n_blocks)));
  CK(cudaMalloc(&P->d_panel_off, sizeof(int64_t) * (n_blocks + 1)));
  CK(cudaMalloc(&P->d_row_ptr, sizeof(int32_t) * (n_blocks + 1)));
  k_bcs_count<<<nbw, 256, 0, st>>>(d_keep, n_shells, P->d_sh_ao0, n_blocks, d_cnt64, P->d_kp, d_k8);
  CK(cudaGetLastError());
  {
    size_t need = 0;
    CK(cub::DeviceScan::ExclusiveSum(nullptr, need, d_cnt64, d_rp64, (int)(n_blocks + 1), st));
    if (need > tmp_bytes) {
      cudaFree(d_tmp);
      d_tmp = nullptr;
      CK(cudaMalloc(&d_tmp, need));
      tmp_bytes = need;
    }
    CK(cub::DeviceScan::ExclusiveSum(d_tmp, tmp_bytes, d_cnt64, d_rp64, (int)(n_blocks + 1), st));
    CK(cub::DeviceScan::ExclusiveSum(d_tmp, tmp_bytes, d_k8, P->d_panel_off, (int)(n_blocks + 1), st));
  }
  int64_t retained = 0;
  CK(cudaMemcpyAsync(&retained, d_rp64 + n_blocks, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
  CK(cudaMemcpyAsync(&P->total_cols, P->d_panel_off + n_blocks, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  if (retained >= ((int64_t)1 << 31) - 4096) {
    set_error("too many retained blocks for int32 BCS indices");
    cleanup();
    return KLDI_EINVAL;
  }
  k_narrow<<<(int)((n_blocks + 1 + 255) / 256), 256, 0, st>>>(d_rp64, n_blocks + 1, P->d_row_ptr);
  CK(cudaGetLastError());
  const int64_t r1 = std::max<int64_t>(1, retained);
  CK(cudaMalloc(&P->d_col_idx, sizeof(int32_t) * r1));
  CK(cudaMalloc(&P->d_blk_col0, sizeof(int32_t) * r1));
  CK(cudaMalloc(&P->d_row_idx, sizeof(int32_t) * r1));
  CK(cudaMalloc(&P->d_pos, sizeof(int32_t) * r1));
  CK(cudaMalloc(&d_erow, sizeof(int32_t) * r1));
  CK(cudaMalloc(&d_eid, sizeof(int32_t) * r1));
  CK(cudaMalloc(&d_skey, sizeof(int32_t) * r1));
  CK(cudaMalloc(&P->d_colidx, sizeof(int32_t) * std::max<int64_t>(1, P->total_cols)));
  CK(cudaMalloc(&P->d_col_ptr, sizeof(int32_t) * (n_shells + 1)));
  CK(cudaMalloc(&d_ccnt, sizeof(int32_t) * (n_shells + 1)));
  CK(cudaMemsetAsync(d_ccnt, 0, sizeof(int32_t) * (n_shells + 1), st));
  k_bcs_fill<<<(int)((n_blocks + 7) / 8), 256, 0, st>>>(d_keep, n_shells, P->d_sh_ao0, n_blocks, P->d_row_ptr,
                                                       P->d_panel_off, P->d_kp, P->d_col_idx, P->d_blk_col0, d_erow,
                                                       d_eid, P->d_colidx, d_ccnt);
  CK(cudaGetLastError());
  {  // BCS(C): col_ptr = inclusive scan of the per-shell counts; entries stably sorted by shell (ascending p inside)
    size_t need = 0;
    CK(cub::DeviceScan::InclusiveSum(nullptr, need, d_ccnt, P->d_col_ptr, n_shells + 1, st));
    size_t need2 = 0;
    int bits = 1;
    while ((1 << bits) < n_shells) ++bits;
    if (retained > 0)
      CK(cub::DeviceRadixSort::SortPairs(nullptr, need2, P->d_col_idx, d_skey, d_eid, P->d_pos, (int)retained, 0, bits,
                                         st));
    need = std::max(need, need2);
    if (need > tmp_bytes) {
      cudaFree(d_tmp);
      d_tmp = nullptr;
      CK(cudaMalloc(&d_tmp, need));
      tmp_bytes = need;
    }
    CK(cub::DeviceScan::InclusiveSum(d_tmp, tmp_bytes, d_ccnt, P->d_col_ptr, n_shells + 1, st));
    if (retained > 0) {
      CK(cub::DeviceRadixSort::SortPairs(d_tmp, tmp_bytes, P->d_col_idx, d_skey, d_eid, P->d_pos, (int)retained, 0,
                                         bits, st));
      k_gather_i32<<<(int)((retained + 255) / 256), 256, 0, st>>>(d_erow, P->d_pos, retained, P->d_row_idx);
      CK(cudaGetLastError());
    }
  }
  // host copies (export, statistics, task list, V schedule)
  row_ptr.assign(n_blocks + 1, 0);
  panel_off.assign(n_blocks + 1, 0);
  col_idx.assign(retained, 0);
  blk_col0.assign(retained, 0);
  row_idx.assign(retained, 0);
  pos.assign(retained, 0);
  col_ptr.assign(n_shells + 1, 0);
#define DH(vec, dptr) \
  if (!(vec).empty()) CK(cudaMemcpyAsync((vec).data(), (dptr), (vec).size() * sizeof((vec)[0]), cudaMemcpyDeviceToHost, st))
  DH(row_ptr, P->d_row_ptr);
  DH(panel_off, P->d_panel_off);
  DH(col_idx, P->d_col_idx);
  DH(blk_col0, P->d_blk_col0);
  DH(row_idx, P->d_row_idx);
  DH(pos, P->d_pos);
  DH(col_ptr, P->d_col_ptr);
  DH(h_kp, P->d_kp);
#undef DH
  CK(cudaStreamSynchronize(st));
  double f_rho_u = 0, f_v_u = 0, f_rho_us = 0;
  int64_t sum_k = 0, max_k = 0;
  for (int64_t p = 0; p < n_blocks; ++p) {
    const int k = h_kp[p];
    if (k > 0) h_tasks.push_back((int32_t)p);
    sum_k += k;
    max_k = std::max<int64_t>(max_k, k);
    f_rho_u += 2.0 * GB * (double)k * k;
    f_rho_us += (double)GB * k * (k + 1.0);
    f_v_u += P->want_grad ? 2.0 * GB * (double)k * k : (double)GB * k * (k + 1.0);
  }
  // S: cost-sorted pull order.  Heavy grid blocks first so that the tail of the persistent kernels is made of light
  // ones; buckets of 96 columns, Morton order kept inside a bucket for the L2 locality of the D gather (measured:
  // cfg1 +2 %, cfg2 +1 %, cfg3 +0.3 % over plain Morton order; fully sorted by K_p loses the locality again).
  constexpr int TASK_BUCKET = 96;
  std::stable_sort(h_tasks.begin(), h_tasks.end(),
                   [&](int32_t a, int32_t b) { return h_kp[a] / TASK_BUCKET > h_kp[b] / TASK_BUCKET; });
  if ((rc = upload(&P->d_tasks, h_tasks, st)) != KLDI_OK) {
    cleanup();
    return rc;
  }
  P->n_tasks = (int32_t)h_tasks.size();
  {
    const kldi_status rcv = vsched_upload(P, h_kp, h_sh_ao0);
    if (rcv != KLDI_OK) {
      cleanup();
      return rcv;
    }
  }
  CK(cudaMalloc(&P->d_blk_amax, sizeof(double) * std::max<int64_t>(1, retained)));
  CK(cudaMemsetAsync(P->d_blk_amax, 0, sizeof(double) * std::max<int64_t>(1, retained), st));

  // ---- P3/P5: tile data.  64 slack columns so that 8-column-padded reads past a panel stay in bounds.
  const size_t tile_bytes = sizeof(double) * GB * (size_t)(P->total_cols + 64);
  CK(cudaMalloc(&P->d_phi, tile_bytes));
  CK(cudaMemsetAsync(P->d_phi, 0, tile_bytes, st));
  CK(cudaMalloc(&P->d_phi_v, tile_bytes));
  CK(cudaMemsetAsync(P->d_phi_v, 0, tile_bytes, st));
  int64_t phi_bytes = 2 * (int64_t)tile_bytes;
  if (P->want_grad) {
    for (int c = 0; c < 3; ++c) {
      CK(cudaMalloc(&P->d_dphi[c], tile_bytes));
      CK(cudaMemsetAsync(P->d_dphi[c], 0, tile_bytes, st));
    }
    CK(cudaMalloc(&P->d_z, tile_bytes));
    CK(cudaMemsetAsync(P->d_z, 0, tile_bytes, st));
    phi_bytes += 4 * (int64_t)tile_bytes;
  }
  if (P->want_grad)
    k_fill<true><<<(int)n_blocks, 128, 0, st>>>(T, P->d_row_ptr, P->d_col_idx, P->d_blk_col0, P->d_panel_off, P->d_gx,
                                                P->d_gy, P->d_gz, P->d_phi, P->d_phi_v, P->d_dphi[0], P->d_dphi[1], P->d_dphi[2],
                                                (unsigned long long*)P->d_blk_amax);
  else
    k_fill<false><<<(int)n_blocks, 128, 0, st>>>(T, P->d_row_ptr, P->d_col_idx, P->d_blk_col0, P->d_panel_off,
                                                 P->d_gx, P->d_gy, P->d_gz, P->d_phi, P->d_phi_v, nullptr, nullptr, nullptr,
                                                 (unsigned long long*)P->d_blk_amax);
  CK(cudaGetLastError());

  // ---- per-call buffers
  const size_t nn = sizeof(double) * (size_t)n_ao * n_ao;
  CK(cudaMalloc(&P->d_Dp, nn));
  CK(cudaMalloc(&P->d_Vp, nn));
  CK(cudaMalloc(&P->d_rho_s, sizeof(double) * n_pad));
  CK(cudaMalloc(&P->d_drho_s, sizeof(double) * 3 * n_pad));
  CK(cudaMalloc(&P->d_wv_s, sizeof(double) * 4 * n_pad));
  CK(cudaMalloc(&P->d_epart, sizeof(double) * (n_blocks + 1)));
  CK(cudaMalloc(&P->d_E, sizeof(double)));
  CK(cudaMalloc(&P->d_ticket, sizeof(int32_t) * 4));
  CK(cudaMallocHost(&P->h_E, sizeof(double)));
  for (auto& e : P->ev) CK(cudaEventCreate(&e));
  CK(cudaStreamSynchronize(st));
  cleanup();
#undef CK
#undef UP

  kldi_stats& S = P->stats;
  S.n_pts = n_pts;
  S.n_blocks = n_blocks;
  S.n_blocks_nonempty = P->n_tasks;
  S.n_ao = n_ao;
  S.n_shells = n_shells;
  S.n_atoms = n_atoms;
  S.want_gradients = P->want_grad;
  S.retained_blocks = retained;
  S.candidate_blocks = n_blocks * (int64_t)n_shells;
  S.sum_k = sum_k;
  S.sum_k_pad = P->total_cols;
  S.max_k = max_k;
  S.phi_bytes = phi_bytes;
  S.workspace_bytes = (int64_t)(2 * nn + sizeof(double) * 8 * n_pad + sizeof(double) * 4 * n_pad +
                                sizeof(int32_t) * (3 * retained * 2 + P->total_cols));
  S.flops_rho_useful = f_rho_u;
  S.flops_rho_useful_sym = f_rho_us;
  S.flops_v_useful = f_v_u;
  S.flops_dense = 2.0 * (double)n_pts * n_ao * n_ao;
  S.eps = P->eps;
  S.plan_seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_start).count();
  return KLDI_OK;
}

}  // namespace kldi
