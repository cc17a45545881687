// H2 on the 5th-generation tensor cores: the LDA rho contraction as int8 slice products with exact int32
// accumulation in tensor memory (the paper's low-precision Tensor-Core block multiplier,
// PAPER.md:218-226, 499-501 App. A-E, with error compensation).  sm_100a: tcgen05.mma kind::i8 (SASS UTCIMMA),
// TMEM accumulators, operands in shared memory, mbarrier pipeline.  KLDI_OPT_RHO_TC.
//
// Arithmetic.  Per grid block p with packed retained columns L(p):
//     X' = Phi_p D'[L,L],  rho = 2 rowsum(Phi_p o X')        D' = lower triangle of D, diagonal halved
// Both operands are split into NSL signed 8-bit digits of base 256 (an error-free transformation of the value rounded
// to 8 NSL bits below its scale):
//     Phi(g,k) ~ sigma_g  sum_i a_i(g,k) 256^-(i+1),   sigma_g = max_k |Phi(g,k)| * 256/127   (row scale, plan time)
//     D'(k,n)  ~ tau_n    sum_j b_j(k,n) 256^-(j+1),   tau_n   = max_k |D'(k,n)|  * 256/127   (column scale, per call)
// The digit pairs of equal weight c = i + j accumulate exactly in one int32 TMEM accumulator (|sum| <= K (c+1) 127^2 <
// 2^31 for K <= 16384), classes c <= NSL-1 are kept (the dropped ones are below 256^-(NSL+1) relative to sigma tau K):
//     X'(g,n) = sigma_g tau_n 256^-(NSL+1)  sum_c acc_c(g,n) 256^(NSL-1-c)
// and the epilogue forms rho in FP64 from the integer recombination and the FP64 Phi columns of the tile.  NSL = 5: 15 int8 products,
// max|d rho| ~ 1e-10 on the 8-water case (tolerance 1e-9); NSL = 6: 21 products, ~3e-13.
#include <cstdio>
#include <cstdlib>

#include "kldi_internal.h"
#include "ptx.cuh"

namespace kldi {
namespace tc {

constexpr int KC = 32;                       // K per tcgen05.mma kind::i8 = packed columns per ring stage
constexpr int NT = 96;                       // N-tile width (NSL * NT <= 512 TMEM columns for NSL = 5)
constexpr int A_SLICE = GB * KC;             // 4096 B: one digit plane of a 128 x 32 Phi chunk
constexpr int NCH = 2 * (NT / 32);           // gather units of a stage (32 columns x 16 K rows) = gather warps per group
constexpr int B_SLICE = (NT / 8) * 256;      // 3072 B: one digit plane of a 32 x 96 D' tile
constexpr int NST = 3;                       // ring stages
constexpr int NGRP = 2;                      // gather groups (alternate stages)
constexpr int NEPI = 8;                      // epilogue warps: NEPI/4 per TMEM lane quarter, 8-column groups dealt round-robin
constexpr int NSET = NEPI / 4;
constexpr int W_PROD = 0, W_MMA = 1, W_GATHER0 = 2, W_EPI0 = W_GATHER0 + NGRP * NCH;  // warp roles
constexpr int NWARPS = W_EPI0 + NEPI;
constexpr int NTHREADS = 32 * NWARPS;        // 704
enum { F_FIRST = 1, F_LAST_TILE = 2, F_LAST_PANEL = 4, F_DONE = 8 };

template <int NSL>
struct Cfg {
  static constexpr int STAGE_BYTES = NSL * (A_SLICE + B_SLICE);
  static constexpr int OFF_EPI = NST * STAGE_BYTES;                   // FP64 Phi columns of the tile (epilogue), [NT][128]
  static constexpr int EPI_BYTES = NT * GB * 8;
  static constexpr int OFF_HDR = OFF_EPI + EPI_BYTES;                 // [NST][4] int
  static constexpr int OFF_KIDX = OFF_HDR + NST * 16;                 // [NST][32] int: plan AO index of the stage's K rows
  static constexpr int OFF_CIDX = OFF_KIDX + NST * KC * 4;            // [4][NT] int: plan AO index of the tile's columns
  static constexpr int OFF_BAR = OFF_CIDX + 4 * NT * 4;               // hdr_full, full_a, full_b, empty [NST]; tmem_full, tmem_empty, epi_full, epi_empty
  static constexpr int OFF_TMEM = OFF_BAR + (4 * NST + 4) * 8;
  static constexpr int OFF_TAU = (OFF_TMEM + 16 + 15) & ~15;          // [NEPI epilogue warps][NT] double
  static constexpr int OFF_RED = OFF_TAU + NEPI * NT * 8;             // [NSET-1][128] double: partial row sums of the other warp sets
  static constexpr int SMEM_BYTES = OFF_RED + (NSET - 1) * GB * 8;
  static constexpr int TMEM_COLS = 512;
  static_assert(NSL * NT <= 512, "accumulator classes do not fit tensor memory");
  static_assert(SMEM_BYTES <= 227 * 1024, "shared memory");
};

// Digit plane of a 128 x 32 Phi chunk, K-major core matrices (8 rows x 16 consecutive K bytes = 128 contiguous bytes):
// the 16 digits of one grid row and 16 consecutive columns are ONE 16-byte word, which is what the epilogue (one lane =
// one grid row) reads back.  Descriptor strides: 128 B between the two K halves (lbo), 256 B between 8-row groups (sbo).
__host__ __device__ __forceinline__ int plane_off_a(int m, int k) {
  return (m >> 3) * 256 + (k >> 4) * 128 + (m & 7) * 16 + (k & 15);
}
// Digit plane of a 32 x 96 D' tile: the same K-major core matrices with the tile column n as the row: a gather lane
// (one column, 16 consecutive K rows) writes ONE 16-byte word per plane.

// ------------------------------------------------------------------------------------------------ plan side
// Digit planes of Phi: per grid block the row scales sigma_g, then for every chunk of 32 packed columns NSL planes of
// 4 KB in the shared-memory image the tensor core reads (so that a ring stage is ONE bulk copy).
template <int NSL>
__global__ void __launch_bounds__(128) k_slice_phi(const int32_t* __restrict__ tasks, const int32_t* __restrict__ kp,
                                                   const int64_t* __restrict__ panel_off,
                                                   const int64_t* __restrict__ chunk_off, const double* __restrict__ phi,
                                                   double* __restrict__ sigma, unsigned char* __restrict__ phiq) {
  __shared__ __align__(16) unsigned char tile[NSL * A_SLICE];
  const int p = tasks[blockIdx.x], g = threadIdx.x;
  const int K8 = (kp[p] + 7) & ~7;
  const int64_t base = panel_off[p];
  double mx = 0.0;
  for (int k = 0; k < K8; ++k) mx = fmax(mx, fabs(phi[(base + k) * GB + g]));
  const double sg = mx > 0.0 ? mx * (256.0 / 127.0) : 1.0;
  sigma[(int64_t)p * GB + g] = sg;
  const double inv = scalbn(1.0 / sg, 8 * NSL);
  const int nchunk = (K8 + KC - 1) / KC;
  for (int c = 0; c < nchunk; ++c) {
    for (int kk = 0; kk < KC; ++kk) {
      const int k = c * KC + kk;
      long long n = 0;
      if (k < K8) n = __double2ll_rn(phi[(base + k) * GB + g] * inv);
#pragma unroll
      for (int i = NSL - 1; i >= 0; --i) {  // balanced base-256 digits, least significant first
        const int d = (int)(signed char)(n & 0xff);
        tile[i * A_SLICE + plane_off_a(g, kk)] = (unsigned char)d;
        n = (n - d) >> 8;
      }
    }
    __syncthreads();
    uint4* dst = reinterpret_cast<uint4*>(phiq + (chunk_off[p] + c) * (int64_t)(NSL * A_SLICE));
    const uint4* src = reinterpret_cast<const uint4*>(tile);
    for (int i = threadIdx.x; i < NSL * A_SLICE / 16; i += 128) dst[i] = src[i];
    __syncthreads();
  }
}

// ------------------------------------------------------------------------------------------------ per call
// tau_n = max_k |D'(k,n)| * 256/127 over the stored (lower-triangular, plan-order) D'.  Non-negative doubles order like
// their bit patterns, so the column maximum is an integer atomicMax.
__global__ void __launch_bounds__(256) k_colmax(const double* __restrict__ Dp, int n, unsigned long long* __restrict__ mx,
                                                int tri) {
  const int j = blockIdx.x * 32 + (threadIdx.x & 31);
  const int r0 = blockIdx.y * 256 + (threadIdx.x >> 5);
  if (j >= n || (tri && blockIdx.y * 256 + 255 < blockIdx.x * 32)) return;  // tri: rows above the diagonal hold zeros
  double m = 0.0;
  for (int r = r0; r < min(n, blockIdx.y * 256 + 256); r += 8) m = fmax(m, fabs(Dp[(int64_t)r * n + j]));
  if (m > 0.0) atomicMax(mx + j, (unsigned long long)__double_as_longlong(m));
}

// Dq[k][n] = the NSL digits of D'(k,n) / tau_n packed in one 64-bit word (byte i = digit i, most significant first);
// tau[n] is rewritten in place from the maximum to the scale.
template <int NSL>
__global__ void __launch_bounds__(256) k_slice_D(const double* __restrict__ Dp, int n, const double* __restrict__ cmax,
                                                 double* __restrict__ tau, unsigned long long* __restrict__ Dq, int tri) {
  const int j = blockIdx.x * 256 + threadIdx.x, i = blockIdx.y;
  if (j >= n) return;
  // tri: strictly above the diagonal Dq was zeroed and is never written (a full-D call marks it dirty, tc_slice_D)
  if (tri && blockIdx.x * 256 > i && i > 0) return;
  const double m = cmax[j];
  const double t = m > 0.0 ? m * (256.0 / 127.0) : 1.0;
  if (i == 0) tau[j] = t;
  unsigned long long q = 0;
  if (!tri || j <= i) {
    long long v = __double2ll_rn(Dp[(int64_t)i * n + j] * scalbn(1.0 / t, 8 * NSL));
#pragma unroll
    for (int s = NSL - 1; s >= 0; --s) {
      const int d = (int)(signed char)(v & 0xff);
      q |= (unsigned long long)(unsigned char)d << (8 * s);
      v = (v - d) >> 8;
    }
  }
  Dq[(int64_t)i * n + j] = q;
}

// ------------------------------------------------------------------------------------------------ the contraction
// Persistent, one CTA per SM, warp-specialised (22 warps):
//   warp 0      scheduler + A producer: pulls grid blocks from the atomic ticket, walks the block's
//               (N-tile, K-chunk) stages, writes the stage header and the AO indices of the stage's K rows (and, per
//               tile, of its columns), bulk-copies the chunk's NSL digit planes of Phi (one 20 KB copy), and after the
//               last stage of a tile the tile's FP64 Phi columns (contiguous in the store: one copy) for the epilogue
//   warps 2-13  B builders, two groups of six on alternate stages: a warp gathers 32 tile columns x 16 K rows of D'
//               (lane = column; an instruction reads ONE row of Dq at the ascending AO indices of 32 consecutive packed
//               columns, a few 128-byte lines), transposes the bytes of the 8-byte digit words to digit planes with PRMT
//               and stores them K-major (NSL x 16-byte stores, conflict-free)
//   warp 1      TMEM owner and MMA issuer: one elected lane issues the tcgen05.mma of a stage and commits them to the
//               stage's empty barrier (and to tmem_full after the last chunk of a tile).  Full-width chunks pair the
//               digit planes of D' (A_i x [B_j | B_j+1] -> classes i+j, i+j+1: 9 instructions), narrow ones use the
//               NSL(NSL+1)/2 single products at N = the columns the chunk reaches
//   warps 14-21 epilogue: TMEM -> registers (one lane = one grid row, two warps per lane quarter on alternate 8-column
//               groups), integer recombination of the classes, FP64 rho += tau_n Phi(g,n) X_int(g,n) with Phi from the
//               staged columns; rho_p at the end of the panel (the two warp sets summed in a fixed order)
// D' is lower triangular in packed order, so only the chunks k0 >= n0 reach tile [n0, n0+Wj) and chunk [k0, k0+32)
// only its columns n < k0 + 32; the chunks are walked in DESCENDING k0, so the first one is full width and overwrites
// (zeroes) every accumulator column of the tile.  The five accumulator classes of a 96-column tile fill tensor memory
// (480 of 512 columns), so the MMAs of a tile and the epilogue of the previous one alternate.
template <int NSL, bool XOUT>
__global__ void __launch_bounds__(NTHREADS, 1)
    k_rho_i8(const int32_t* __restrict__ tasks, int n_tasks, int32_t* __restrict__ ticket, const int32_t* __restrict__ kp,
             const int64_t* __restrict__ panel_off, const int64_t* __restrict__ chunk_off,
             const int32_t* __restrict__ colidx, const double* __restrict__ phi, const unsigned char* __restrict__ phiq,
             const double* __restrict__ sigma, const unsigned long long* __restrict__ Dq, const double* __restrict__ tau,
             int n_ao, double* __restrict__ rho_s, double* __restrict__ x_out, long long* __restrict__ dbg) {
  using C = Cfg<NSL>;
  extern __shared__ __align__(128) unsigned char smem[];
  long long tw[6] = {0, 0, 0, 0, 0, 0};  // debug: cycles spent in the waits of this warp's role
  auto twait = [&](int slot, uint32_t bar, uint32_t parity) {
    if (dbg) {
      const long long t0 = clock64();
      mbar_wait(bar, parity);
      tw[slot] += clock64() - t0;
    } else {
      mbar_wait(bar, parity);
    }
  };
  const long long t_begin = dbg ? clock64() : 0;
  volatile int* hdr = reinterpret_cast<volatile int*>(smem + C::OFF_HDR);
  volatile int* kidx = reinterpret_cast<volatile int*>(smem + C::OFF_KIDX);
  volatile int* cidx = reinterpret_cast<volatile int*>(smem + C::OFF_CIDX);
  const uint32_t bar0 = smem_u32(smem + C::OFF_BAR);
  const uint32_t b_hdr = bar0, b_fa = bar0 + 8 * NST, b_fb = bar0 + 16 * NST, b_empty = bar0 + 24 * NST;
  const uint32_t b_tfull = bar0 + 32 * NST, b_tempty = b_tfull + 8, b_efull = b_tfull + 16, b_eempty = b_tfull + 24;
  volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(smem + C::OFF_TMEM);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid == 0) {
    for (int s = 0; s < NST; ++s) {
      mbar_init(b_hdr + 8 * s, 1);
      mbar_init(b_fa + 8 * s, 1);
      mbar_init(b_fb + 8 * s, NCH);
      mbar_init(b_empty + 8 * s, 1 + NEPI);  // tcgen05.commit of the stage's MMAs + the epilogue warps (header read)
    }
    mbar_init(b_tfull, 1);
    mbar_init(b_tempty, NEPI);
    mbar_init(b_efull, 1);
    mbar_init(b_eempty, NEPI);
    fence_mbar_init();
  }
  if (warp == W_MMA) tmem_alloc(smem_u32(smem + C::OFF_TMEM), C::TMEM_COLS);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;

  if (warp == W_PROD) {
    // ------------------------------------------------------------------ scheduler + A producer
    uint32_t t = 0;     // stage sequence number: slot t % NST, use t / NST
    uint32_t tile = 0;  // tile sequence number
    for (;;) {
      int task = 0;
      if (lane == 0) task = atomicAdd(ticket, 1);
      task = __shfl_sync(0xffffffffu, task, 0);
      if (task >= n_tasks) break;
      const int p = tasks[task];
      const int K8 = (kp[p] + 7) & ~7, K32 = (K8 + KC - 1) & ~(KC - 1);
      const int64_t base = panel_off[p], cbase = chunk_off[p];
      const int ntile = (K32 + NT - 1) / NT;
      const int W = ((K32 / KC + ntile - 1) / ntile) * KC;  // tiles start on chunk boundaries
      for (int jt = 0; jt < ntile; ++jt, ++tile) {
        const int n0 = jt * W, Wj = min(W, K32 - n0);
        int cn[NT / 32];
#pragma unroll
        for (int u = 0; u < NT / 32; ++u) {
          const int n = n0 + lane + 32 * u;
          cn[u] = (lane + 32 * u < Wj && n < K8) ? colidx[base + n] : -1;
        }
        // XOUT (X = A D with the FULL D, the X builds of the nuclear gradient): every chunk reaches every tile
        const int kmin = XOUT ? 0 : n0;
        for (int k0 = K32 - KC; k0 >= kmin; k0 -= KC) {
          const int s = t % NST;
          const int k = k0 + lane;
          const int kr = k < K8 ? colidx[base + k] : -1;
          if (t >= NST) twait(0, b_empty + 8 * s, ((t / NST) - 1) & 1);
          kidx[s * KC + lane] = kr;
          if (k0 == K32 - KC) {  // a tile's column indices live 4 tiles: every tile has at least one stage
#pragma unroll
            for (int u = 0; u < NT / 32; ++u) cidx[(tile & 3) * NT + lane + 32 * u] = cn[u];
          }
          __syncwarp();
          if (lane == 0) {
            int fl = 0;
            if (k0 == K32 - KC) fl |= F_FIRST;
            if (k0 == kmin) fl |= F_LAST_TILE | (jt == ntile - 1 ? F_LAST_PANEL : 0);
            const int wact = XOUT ? Wj : min(Wj, k0 + KC - n0);
            hdr[4 * s + 0] = p;
            hdr[4 * s + 1] = n0 | (k0 << 16);
            hdr[4 * s + 2] = fl | (wact << 8) | (Wj << 16) | ((tile & 3) << 24);
            hdr[4 * s + 3] = K8;
            mbar_arrive(b_hdr + 8 * s);
            mbar_arrive_expect_tx(b_fa + 8 * s, NSL * A_SLICE);
            bulk_g2s(smem_u32(smem + s * C::STAGE_BYTES), phiq + (cbase + k0 / KC) * (int64_t)(NSL * A_SLICE),
                     NSL * A_SLICE, b_fa + 8 * s);
          }
          __syncwarp();
          ++t;
        }
        // (the tile's FP64 Phi columns for its epilogue are fetched by the epilogue warps themselves, see there: the
        // producer never waits for an epilogue and keeps the ring full with the next tile's stages)
      }
    }
    for (int e = 0; e < NGRP; ++e) {  // one DONE stage per gather group (the other roles stop at the first)
      const int s = t % NST;
      if (t >= NST) mbar_wait(b_empty + 8 * s, ((t / NST) - 1) & 1);
      if (lane == 0) {
        hdr[4 * s + 2] = F_DONE;
        mbar_arrive(b_hdr + 8 * s);
      }
      __syncwarp();
      ++t;
    }
  } else if (warp == W_MMA) {
    // ------------------------------------------------------------------ MMA issuer
    uint32_t t = 0, tile = 0;
    uint64_t da[NST], db[NST];
#pragma unroll
    for (int s = 0; s < NST; ++s) {
      da[s] = umma_smem_desc(smem_u32(smem + s * C::STAGE_BYTES), 128, 256);
      db[s] = umma_smem_desc(smem_u32(smem + s * C::STAGE_BYTES + NSL * A_SLICE), 128, 256);
    }
    for (;;) {
      const int s = t % NST;
      const uint32_t ph = (t / NST) & 1;
      twait(0, b_hdr + 8 * s, ph);
      const int h2 = hdr[4 * s + 2];
      if (h2 & F_DONE) break;
      const int wact = (h2 >> 8) & 0xff;
      if ((h2 & F_FIRST) && tile > 0) twait(1, b_tempty, (tile - 1) & 1);  // the epilogue has drained the accumulators
      twait(2, b_fa + 8 * s, ph);
      twait(3, b_fb + 8 * s, ph);
      tc_fence_after();
      if (elect_one()) {
        const uint32_t idesc = umma_idesc_s8(wact);
        const uint32_t keep = (h2 & F_FIRST) ? 0u : 1u;
        uint64_t a = da[0], b = db[0];
#pragma unroll
        for (int q = 1; q < NST; ++q)
          if (s == q) { a = da[q]; b = db[q]; }
        // Full-width chunks: digit i of Phi against the digits j, j+1 of D' in ONE instruction.  The B planes of a stage
        // are contiguous and so are the accumulator classes, so A_i x [B_j | B_j+1] (N = 2 NT) adds into the classes i+j
        // and i+j+1, and the 4 KB A plane is read from shared memory once for two products (9 instructions instead of
        // 15).  The plane rows beyond the tile width only reach accumulator columns nobody reads.  Narrow (diagonal)
        // chunks use single planes at N = wact.
        if (wact == ((h2 >> 16) & 0xff)) {
          const uint32_t id2 = umma_idesc_s8(2 * NT), id1 = umma_idesc_s8(NT);
#pragma unroll
          for (int i = 0; i < NSL; ++i) {
#pragma unroll
            for (int j = 0; i + j < NSL; j += 2) {
              const bool two = i + j + 1 < NSL;
              umma_i8(tmem + (i + j) * NT, a + (uint64_t)(i * (A_SLICE >> 4)), b + (uint64_t)(j * (B_SLICE >> 4)),
                      two ? id2 : id1, i == 0 ? keep : 1u);
            }
          }
        } else {
#pragma unroll
          for (int i = 0; i < NSL; ++i)
#pragma unroll
            for (int j = 0; i + j < NSL; ++j)
              umma_i8(tmem + (i + j) * NT, a + (uint64_t)(i * (A_SLICE >> 4)), b + (uint64_t)(j * (B_SLICE >> 4)), idesc,
                      i == 0 ? keep : 1u);
        }
        umma_commit(b_empty + 8 * s);
        if (h2 & F_LAST_TILE) umma_commit(b_tfull);
      }
      __syncwarp();
      if (h2 & F_LAST_TILE) ++tile;
      ++t;
    }
  } else if (warp < W_EPI0) {
    // ------------------------------------------------------------------ B builders
    // unit of a warp: 32 tile columns (lane = column) x 16 K rows; an instruction reads ONE row of Dq at the 32
    // ascending AO indices of consecutive packed columns, so a warp load touches a few 128-byte lines, not 32
    const int grp = (warp - W_GATHER0) / NCH, c = (warp - W_GATHER0) % NCH;
    const int ng = c >> 1, h = c & 1;
    for (uint32_t t = grp;; t += NGRP) {
      const int s = t % NST;
      const uint32_t ph = (t / NST) & 1;
      twait(0, b_hdr + 8 * s, ph);
      const int h2 = hdr[4 * s + 2];
      if (h2 & F_DONE) break;
      const int wact = (h2 >> 8) & 0xff;
      if (32 * ng < wact) {
        const int cj = cidx[((h2 >> 24) & 3) * NT + 32 * ng + lane];
        const unsigned long long* col = Dq + max(cj, 0);
        unsigned long long q[16];
#pragma unroll
        for (int r = 0; r < 16; ++r) {
          const int kr = kidx[s * KC + 16 * h + r];
          q[r] = (kr >= 0 && cj >= 0) ? __ldg(col + (int64_t)kr * n_ao) : 0ull;
        }
        const uint32_t dst = smem_u32(smem + s * C::STAGE_BYTES + NSL * A_SLICE) + (4 * ng + (lane >> 3)) * 256 + h * 128 +
                             (lane & 7) * 16;
        // byte transposition: word w of plane i holds digit i of the K rows 4w .. 4w+3
#pragma unroll
        for (int i0 = 0; i0 < NSL; i0 += 4) {
          uint32_t o[4][4];
#pragma unroll
          for (int w = 0; w < 4; ++w) {
            uint32_t x0, x1, x2, x3;
            if (i0 == 0) {
              x0 = (uint32_t)q[4 * w]; x1 = (uint32_t)q[4 * w + 1]; x2 = (uint32_t)q[4 * w + 2]; x3 = (uint32_t)q[4 * w + 3];
            } else {
              x0 = (uint32_t)(q[4 * w] >> 32); x1 = (uint32_t)(q[4 * w + 1] >> 32);
              x2 = (uint32_t)(q[4 * w + 2] >> 32); x3 = (uint32_t)(q[4 * w + 3] >> 32);
            }
            const uint32_t a = __byte_perm(x0, x1, 0x5140), b = __byte_perm(x2, x3, 0x5140);
            o[0][w] = __byte_perm(a, b, 0x5410);
            o[1][w] = __byte_perm(a, b, 0x7632);
            if (i0 + 2 < NSL) {
              const uint32_t e = __byte_perm(x0, x1, 0x7362), f = __byte_perm(x2, x3, 0x7362);
              o[2][w] = __byte_perm(e, f, 0x5410);
              o[3][w] = __byte_perm(e, f, 0x7632);
            }
          }
#pragma unroll
          for (int i = 0; i < 4; ++i)
            if (i0 + i < NSL)
              asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(dst + (i0 + i) * B_SLICE), "r"(o[i][0]),
                           "r"(o[i][1]), "r"(o[i][2]), "r"(o[i][3])
                           : "memory");
        }
        fence_proxy_async_smem();
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(b_fb + 8 * s);
    }
  } else {
    // ------------------------------------------------------------------ epilogue
    const int qd = warp & 3;                 // TMEM lane quarter of this warp
    const int hs = (warp - W_EPI0) >> 2;     // warp set: 8-column groups with group % NSET == hs
    const int g = 32 * qd + lane;
    double* tau_s = reinterpret_cast<double*>(smem + C::OFF_TAU) + (warp - W_EPI0) * NT;
    double* red = reinterpret_cast<double*>(smem + C::OFF_RED);
    const uint32_t tl = tmem + ((uint32_t)(32 * qd) << 16);
    const double* ephi = reinterpret_cast<const double*>(smem + C::OFF_EPI) + g;  // this row of the tile's Phi columns
    double rs = 0.0;
    uint32_t tile = 0;
    for (uint32_t t = 0;; ++t) {
      const int s = t % NST;
      twait(0, b_hdr + 8 * s, (t / NST) & 1);
      const int h2 = hdr[4 * s + 2];
      if (h2 & F_DONE) break;
      const int p = hdr[4 * s + 0], n0 = hdr[4 * s + 1] & 0xffff, K8 = hdr[4 * s + 3];
      __syncwarp();
      if (lane == 0) mbar_arrive(b_empty + 8 * s);  // header read
      if ((h2 & F_FIRST) && warp == W_EPI0) {
        // first stage of a tile: fetch the tile's FP64 Phi columns for its epilogue (contiguous in the store: ONE bulk
        // copy) as soon as every epilogue warp has left the previous tile (single buffer); it lands during the tile's MMAs
        if (tile > 0) twait(4, b_eempty, (tile - 1) & 1);
        if (lane == 0) {
          const uint32_t bytes = (uint32_t)min((h2 >> 16) & 0xff, K8 - n0) * (GB * 8);
          mbar_arrive_expect_tx(b_efull, bytes);
          bulk_g2s(smem_u32(smem + C::OFF_EPI), phi + (panel_off[p] + n0) * GB, bytes, b_efull);
        }
        __syncwarp();
      }
      if (!(h2 & F_LAST_TILE)) continue;
      const int wj = min((h2 >> 16) & 0xff, K8 - n0);  // real columns of the tile
      const volatile int* cn = cidx + ((h2 >> 24) & 3) * NT;
      for (int j = lane; j < wj; j += 32) tau_s[j] = tau[cn[j]];
      __syncwarp();
      twait(1, b_efull, tile & 1);
      twait(2, b_tfull, tile & 1);
      tc_fence_after();
      const long long t_e0 = dbg ? clock64() : 0;
      double rs2 = 0.0;
      double xs = 0.0;
      double* xg = nullptr;
      if (XOUT) {
        xs = scalbn(sigma[(int64_t)p * GB + g], -8 * (NSL + 1));
        xg = x_out + (panel_off[p] + n0) * GB + g;
      }
      for (int j0 = 8 * hs; j0 < wj; j0 += 8 * NSET) {
        int32_t acc[NSL][8];
#pragma unroll
        for (int c = 0; c < NSL; ++c) tmem_ld8(tl + c * NT + j0, acc[c]);
        double f[8];  // rho form: tau_n Phi(g,n) of the columns j0 .. j0+7; X form: tau_n alone (Phi is read when used)
#pragma unroll
        for (int j = 0; j < 8; ++j) f[j] = tau_s[j0 + j];
        tmem_ld_wait();
#pragma unroll
        for (int j = 0; j < 8; ++j) {
          // X_int = sum_c acc_c 256^(NSL-1-c) in two integer parts below 2^51, each to FP64 through the 2^52 + 2^51
          // mantissa trick (an integer multiply-add chain + one DADD)
          constexpr long long MAGIC = 0x4338000000000000LL;
          constexpr double MAGIC_D = 6755399441055744.0;
          double xd;
          if (NSL == 5) {
            const long long xh = (long long)acc[0][j] * 65536 + ((long long)acc[1][j] * 256 + ((long long)acc[2][j] + MAGIC));
            const long long xl = (long long)acc[3][j] * 256 + ((long long)acc[4][j] + MAGIC);
            xd = fma(__longlong_as_double(xh) - MAGIC_D, 65536.0, __longlong_as_double(xl) - MAGIC_D);
          } else {
            long long x = 0;
#pragma unroll
            for (int c = 0; c < NSL; ++c) x = x * 256 + acc[c][j];
            xd = (double)x;
          }
          const double t = f[j] * xd;
          if (XOUT) xg[(int64_t)(j0 + j) * GB] = xs * t;  // X(g,n): 256 B per warp and column
          if (j & 1)
            rs2 = fma(ephi[(j0 + j) * GB], t, rs2);
          else
            rs = fma(ephi[(j0 + j) * GB], t, rs);
        }
      }
      rs += rs2;
      tc_fence_before();
      __syncwarp();
      if (lane == 0) {
        mbar_arrive(b_tempty);
        mbar_arrive(b_eempty);
      }
      if (dbg) tw[3] += clock64() - t_e0;
      ++tile;
      if (h2 & F_LAST_PANEL) {  // the warp sets of a row: sets 1.. through shared memory, summed in a fixed order
        if (hs > 0) red[(hs - 1) * GB + g] = rs;
        asm volatile("bar.sync 1, %0;" ::"n"(32 * NEPI) : "memory");
        if (hs == 0) {
          const double sg = sigma[(int64_t)p * GB + g];
#pragma unroll
          for (int q = 0; q < NSET - 1; ++q) rs += red[q * GB + g];
          rho_s[(int64_t)p * GB + g] = (XOUT ? 1.0 : 2.0) * sg * scalbn(rs, -8 * (NSL + 1));
        }
        asm volatile("bar.sync 1, %0;" ::"n"(32 * NEPI) : "memory");
        rs = 0.0;
      }
    }
  }
  if (dbg && lane == 0) {  // per role: [0..5] wait slots, [6] lifetime, [7] warps
    const int role = warp == W_PROD ? 0 : warp == W_MMA ? 1 : warp < W_EPI0 ? 2 : 3;
    for (int i = 0; i < 6; ++i) atomicAdd(reinterpret_cast<unsigned long long*>(dbg + 8 * role + i), (unsigned long long)tw[i]);
    atomicAdd(reinterpret_cast<unsigned long long*>(dbg + 8 * role + 6), (unsigned long long)(clock64() - t_begin));
    atomicAdd(reinterpret_cast<unsigned long long*>(dbg + 8 * role + 7), 1ull);
  }
  tc_fence_before();
  __syncthreads();
  if (warp == W_MMA) tmem_dealloc(tmem, C::TMEM_COLS);
}

}  // namespace tc

// ------------------------------------------------------------------------------------------------ host side
template <int NSL>
static kldi_status tc_prepare(kldi_plan* P) {
  if (P->d_chunk_off) return KLDI_OK;
  if (P->stats.max_k > 16384) {
    set_error("KLDI_OPT_RHO_TC: a grid block retains %lld AO columns; the int32 accumulators hold 16384", (long long)P->stats.max_k);
    return KLDI_ESTATE;
  }
  std::vector<int64_t> h_chunk(P->n_blocks + 1, 0);
  for (int64_t p = 0; p < P->n_blocks; ++p) {
    const int64_t k8 = P->h_panel_off[p + 1] - P->h_panel_off[p];
    h_chunk[p + 1] = h_chunk[p] + (k8 + tc::KC - 1) / tc::KC;
  }
  P->tc_chunks = h_chunk[P->n_blocks];
  {  // int8 operations the contraction issues (mirrors the producer / MMA issuer loops of k_rho_i8)
    double ops = 0.0;
    const int npair = NSL * (NSL + 1) / 2;
    for (int64_t p = 0; p < P->n_blocks; ++p) {
      const int k8 = (int)(P->h_panel_off[p + 1] - P->h_panel_off[p]);
      if (!k8) continue;
      const int K32 = (k8 + tc::KC - 1) & ~(tc::KC - 1), ntile = (K32 + tc::NT - 1) / tc::NT;
      const int W = ((K32 / tc::KC + ntile - 1) / ntile) * tc::KC;
      for (int jt = 0; jt < ntile; ++jt) {
        const int n0 = jt * W, Wj = std::min(W, K32 - n0);
        for (int k0 = K32 - tc::KC; k0 >= n0; k0 -= tc::KC) {
          const int wact = std::min(Wj, k0 + tc::KC - n0);
          // full-width chunks pair the D' planes at the tile pitch NT (plane rows beyond Wj are issued too)
          ops += 2.0 * GB * tc::KC * npair * (wact == Wj ? tc::NT : wact);
        }
      }
    }
    P->stats.ops_rho_tc = ops;
  }
  KLDI_CUDA(cudaMalloc(&P->d_Dq, sizeof(unsigned long long) * (size_t)P->n_ao * P->n_ao));
  KLDI_CUDA(cudaMemsetAsync(P->d_Dq, 0, sizeof(unsigned long long) * (size_t)P->n_ao * P->n_ao, P->stream));
  KLDI_CUDA(cudaMalloc(&P->d_tau, sizeof(double) * 2 * P->n_ao));
  KLDI_CUDA(cudaMalloc(&P->d_chunk_off, sizeof(int64_t) * (P->n_blocks + 1)));
  KLDI_CUDA(cudaMemcpyAsync(P->d_chunk_off, h_chunk.data(), sizeof(int64_t) * (P->n_blocks + 1), cudaMemcpyHostToDevice, P->stream));
  KLDI_CUDA(cudaStreamSynchronize(P->stream));  // h_chunk goes out of scope
  kldi_status rc = ensure_smem_attr((const void*)tc::k_rho_i8<NSL, false>, tc::Cfg<NSL>::SMEM_BYTES, P->device);
  if (rc != KLDI_OK) return rc;
  return ensure_smem_attr((const void*)tc::k_rho_i8<NSL, true>, tc::Cfg<NSL>::SMEM_BYTES, P->device);
}

// Digit planes and row scales of one store of the rho layout (Phi or a gradient store), once per plan.
template <int NSL>
static kldi_status tc_prepare_store(kldi_plan* P, const double* store, unsigned char** planes, double** scales) {
  if (*planes) return KLDI_OK;
  KLDI_CUDA(cudaMalloc(scales, sizeof(double) * P->n_pad));
  KLDI_CUDA(cudaMalloc(planes, (size_t)std::max<int64_t>(1, P->tc_chunks) * NSL * tc::A_SLICE));
  if (P->n_tasks > 0) {
    tc::k_slice_phi<NSL><<<P->n_tasks, 128, 0, P->stream>>>(P->d_tasks, P->d_kp, P->d_panel_off, P->d_chunk_off, store,
                                                           *scales, *planes);
    KLDI_LAUNCHED(P);
  }
  P->stats.phi_bytes += (int64_t)P->tc_chunks * NSL * tc::A_SLICE;
  return KLDI_OK;
}

// The digits and column scales of the matrix in P->d_Dp, once per call: tri = D' (lower triangle, diagonal halved; only
// that triangle of Dq is written, the rest stays zero) or the full D (the X builds of the nuclear gradient).
template <int NSL>
static kldi_status tc_slice_D(kldi_plan* P, bool tri = true) {
  const int n = P->n_ao;
  if (tri && P->dq_upper_dirty)  // a full-D call has written the upper triangle: back to zero for the triangular form
    KLDI_CUDA(cudaMemsetAsync(P->d_Dq, 0, sizeof(unsigned long long) * (size_t)n * n, P->stream));
  P->dq_upper_dirty = !tri;
  double* cmax = P->d_tau + n;
  KLDI_CUDA(cudaMemsetAsync(cmax, 0, sizeof(double) * n, P->stream));
  tc::k_colmax<<<dim3((n + 31) / 32, (n + 255) / 256), 256, 0, P->stream>>>(P->d_Dp, n, reinterpret_cast<unsigned long long*>(cmax), tri ? 1 : 0);
  KLDI_LAUNCHED(P);
  tc::k_slice_D<NSL><<<dim3((n + 255) / 256, n), 256, 0, P->stream>>>(P->d_Dp, n, cmax, P->d_tau, P->d_Dq, tri ? 1 : 0);
  KLDI_LAUNCHED(P);
  return KLDI_OK;
}

// out_s[g] = 2 sum_{mu >= nu} D'_{mu,nu} A_{g,mu} A_{g,nu} for the store A (FP64 columns `store`, digit planes `planes`)
// XOUT: the full-D form, out_s[g] = sum_{mu,nu} D_{mu,nu} A_{g,mu} A_{g,nu} and x_out = A D (rho layout)
template <int NSL, bool XOUT = false>
static kldi_status tc_contract(kldi_plan* P, const double* store, const unsigned char* planes, const double* scales,
                               double* out_s, double* x_out = nullptr) {
  KLDI_CUDA(cudaMemsetAsync(out_s, 0, sizeof(double) * P->n_pad, P->stream));
  KLDI_CUDA(cudaMemsetAsync(P->d_ticket, 0, sizeof(int32_t) * 4, P->stream));
  const int grid = P->n_sm < P->n_tasks ? P->n_sm : P->n_tasks;
  static const bool debug = getenv("KLDI_TC_DEBUG") != nullptr;  // per-role wait cycles, printed to stderr (synchronises)
  long long* dbg = nullptr;
  if (debug) {
    KLDI_CUDA(cudaMalloc(&dbg, 32 * sizeof(long long)));
    KLDI_CUDA(cudaMemsetAsync(dbg, 0, 32 * sizeof(long long), P->stream));
  }
  tc::k_rho_i8<NSL, XOUT><<<grid, tc::NTHREADS, tc::Cfg<NSL>::SMEM_BYTES, P->stream>>>(
      P->d_tasks, P->n_tasks, P->d_ticket, P->d_kp, P->d_panel_off, P->d_chunk_off, P->d_colidx, store, planes, scales,
      P->d_Dq, P->d_tau, P->n_ao, out_s, x_out, dbg);
  KLDI_LAUNCHED(P);
  if (debug) {
    long long h[32];
    KLDI_CUDA(cudaStreamSynchronize(P->stream));
    KLDI_CUDA(cudaMemcpy(h, dbg, sizeof(h), cudaMemcpyDeviceToHost));
    cudaFree(dbg);
    const char* names[4] = {"producer [empty, epi_empty]", "mma [hdr, tmem_empty, full_a, full_b]", "gather [hdr]",
                            "epilogue [hdr, epi_full, tmem_full, compute]"};
    for (int r = 0; r < 4; ++r) {
      const double w = (double)h[8 * r + 7];
      fprintf(stderr, "k_rho_i8 %-46s warps %4.0f life %9.0f waits", names[r], w, h[8 * r + 6] / w);
      for (int i = 0; i < 4; ++i) fprintf(stderr, " %9.0f", h[8 * r + i] / w);
      fprintf(stderr, "  (cycles per warp)\n");
    }
  }
  return KLDI_OK;
}

constexpr int TC_NSL = 5;

// rho_s of every grid block from D' in P->d_Dp (written by launch_permute_D in its triangular form).
kldi_status launch_rho_tc(kldi_plan* P) {
  kldi_status rc = tc_prepare<TC_NSL>(P);
  if (rc != KLDI_OK) return rc;
  if ((rc = tc_prepare_store<TC_NSL>(P, P->d_phi, &P->d_phiq, &P->d_sigma)) != KLDI_OK) return rc;
  if (P->n_tasks == 0) {
    KLDI_CUDA(cudaMemsetAsync(P->d_rho_s, 0, sizeof(double) * P->n_pad, P->stream));
    return KLDI_OK;
  }
  if ((rc = tc_slice_D<TC_NSL>(P)) != KLDI_OK) return rc;
  return tc_contract<TC_NSL>(P, P->d_phi, P->d_phiq, P->d_sigma, P->d_rho_s);
}

// The three LDA-form builds of the kinetic-energy density on the gradient stores, D' split once.
kldi_status launch_tau_tc(kldi_plan* P) {
  kldi_status rc = tc_prepare<TC_NSL>(P);
  if (rc != KLDI_OK) return rc;
  for (int c = 0; c < 3; ++c)
    if ((rc = tc_prepare_store<TC_NSL>(P, P->d_dphi[c], &P->d_dphiq[c], &P->d_dsigma[c])) != KLDI_OK) return rc;
  if (P->n_tasks == 0) {
    KLDI_CUDA(cudaMemsetAsync(P->d_drho_s, 0, sizeof(double) * 3 * P->n_pad, P->stream));
    return KLDI_OK;
  }
  if ((rc = tc_slice_D<TC_NSL>(P)) != KLDI_OK) return rc;
  for (int c = 0; c < 3; ++c)
    if ((rc = tc_contract<TC_NSL>(P, P->d_dphi[c], P->d_dphiq[c], P->d_dsigma[c], P->d_drho_s + (size_t)c * P->n_pad)) !=
        KLDI_OK)
      return rc;
  return KLDI_OK;
}

// X = A D with the FULL D (already in P->d_Dp) for the store A = Phi (which = 0) or d_c Phi (which = 1 + c), written to
// x_out in the rho layout; rho_out gets rowsum(A o X).  slice_d: split D into digits first (once per call).
kldi_status launch_x_tc(kldi_plan* P, int which, double* x_out, double* rho_out, bool slice_d) {
  kldi_status rc = tc_prepare<TC_NSL>(P);
  if (rc != KLDI_OK) return rc;
  const double* store = which == 0 ? P->d_phi : P->d_dphi[which - 1];
  unsigned char** planes = which == 0 ? &P->d_phiq : &P->d_dphiq[which - 1];
  double** scales = which == 0 ? &P->d_sigma : &P->d_dsigma[which - 1];
  if ((rc = tc_prepare_store<TC_NSL>(P, store, planes, scales)) != KLDI_OK) return rc;
  if (P->n_tasks == 0) {
    KLDI_CUDA(cudaMemsetAsync(rho_out, 0, sizeof(double) * P->n_pad, P->stream));
    return KLDI_OK;
  }
  if (slice_d && (rc = tc_slice_D<TC_NSL>(P, false)) != KLDI_OK) return rc;
  return tc_contract<TC_NSL, true>(P, store, *planes, *scales, rho_out, x_out);
}

}  // namespace kldi
