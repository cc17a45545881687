// Per-evaluation kernels of libkldi (the hot path).  sm_100a, FP64.
//   H1 k_permute_D   — D in plan AO order
//   H2 k_rho         — X_p = Phi_p D[L(p),L(p)], rho_p = rowsum(Phi_p o X_p) (Eq. 4/18)
//   H3 k_xc          — Slater / PBE-x per point, wv = w v, deterministic energy reduction (Eq. 1/3)
//   H4 k_vgram       — G_p = Phi_p^T diag(wv_p) Phi_p scattered into V (Eq. 5/16): vgram.cu
//   H5 k_finalise_V  — mirror / symmetrise, back to caller AO order
//   F2 k_grad_cols   — LDA nuclear-gradient contraction from the X store k_rho writes
//   F4 k_tau_combine — kinetic-energy density from three LDA-form k_rho builds on the gradient stores (§8(f4))
// H2 and H4 are persistent, warp-specialised kernels: producer warps pull grid-block tasks from an atomic
// ticket (the paper's pull-based pool, on-device) and stream operand tiles through an mbarrier
// ring with bulk-async copies (TMA engine) and 8-byte cp.async; 16 (k_rho) / 15 (k_vgram) consumer warps issue
// FP64 tensor-core MMAs (DMMA.8x8x4) on register accumulators.
#include <cstdio>

#include "ao_eval.cuh"
#include "kldi_internal.h"
#include "ptx.cuh"

namespace kldi {

constexpr int LD = GB + 4;  // padded smem leading dimension of a 128-row column: conflict-free 8-B fragments

// ===================================================================================== H1
// TRI: the strictly lower triangle of D (plan order), the diagonal halved, zeros above.  D is symmetric, so
// rho = sum_{mu,nu} D_{mu nu} chi_mu chi_nu = 2 sum_{mu >= nu} D'_{mu nu} chi_mu chi_nu: the rho contraction then
// only visits the block pairs on one side of the diagonal (the symmetry of PAPER.md:220).
template <bool TRI>
__global__ void k_permute_D(const double* __restrict__ D, const int32_t* __restrict__ ao_perm, int n,
                            double* __restrict__ Dp) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x, i = blockIdx.y;
  if (j >= n) return;
  double v = 0.0;
  if (!TRI || j <= i) {
    // D is symmetric (kldi.h): always read its lower triangle, so that kldi_exc_host only has to upload that half
    const int a = ao_perm[i], b = ao_perm[j];
    v = D[(int64_t)max(a, b) * n + min(a, b)];
    if (TRI && j == i) v *= 0.5;
  }
  Dp[(int64_t)i * n + j] = v;
}

// ===================================================================================== H2
namespace rho {
constexpr int NST = 3;                    // ring stages
constexpr int KC = 32;                    // packed columns (K) per stage
constexpr int NT = 128;                   // max N-tile width
constexpr int PHI_BYTES = KC * LD * 8;    // 33,792
constexpr int D_BYTES = KC * (NT + 4) * 8;  // 33,792
constexpr int STAGE_BYTES = PHI_BYTES + D_BYTES;
constexpr int SMEM_BYTES = NST * STAGE_BYTES + NST * 16 + 2 * NST * 8 + 16;
constexpr int NCW = 16;                   // consumer warps: 8 grid rows each, all N columns
constexpr int NPW = 4;                    // producer warps: each stages 8 of the 32 chunk rows
constexpr int NTHREADS = 32 * (NCW + NPW);
enum { F_FIRST = 1, F_LAST_TILE = 2, F_LAST_PANEL = 4, F_DONE = 8, F_EPI = 16 };
constexpr int EC = 16;                    // GGA epilogue stage: 16 tile columns of Phi, dxPhi, dyPhi, dzPhi
}  // namespace rho

// One ring stage of a consumer warp (8 grid rows x all N columns): nks k-steps of 4, NJ active 8-column groups
// (compile-time, so that no MMA is predicated: a predicated mma.sync costs a WARPSYNC + NOP pair around every
// DMMA).  B fragments are loaded 8 at a time to stay inside the 96-register budget of 20 warps per SM.
template <int NJ>
__device__ __forceinline__ void rho_ksteps(double (&acc)[16][2], const double* __restrict__ ps,
                                           const double* __restrict__ ds, int nks) {
#pragma unroll 2
  for (int ks = 0; ks < nks; ++ks) {
    const double a = ps[ks * 4 * LD];
#pragma unroll
    for (int j0 = 0; j0 < NJ; j0 += 8) {
      double b[8];
#pragma unroll
      for (int j = 0; j < 8; ++j)
        if (j0 + j < NJ) b[j] = ds[ks * 4 * (rho::NT + 4) + 8 * (j0 + j)];
#pragma unroll
      for (int j = 0; j < 8; ++j)
        if (j0 + j < NJ) dmma884(acc[j0 + j][0], acc[j0 + j][1], a, b[j]);
    }
  }
}

// TRI, the chunk's own (up to 4) column groups J0..: that 32x32 block of D' is itself lower triangular, so the
// k-steps 2m, 2m+1 (chunk rows 8m..8m+7) only reach the own groups jj <= m -- 20 DMMAs instead of 32.
template <int J0>
__device__ __forceinline__ void rho_diag(double (&acc)[16][2], const double* __restrict__ ps,
                                         const double* __restrict__ ds, int nown) {
#pragma unroll
  for (int m = 0; m < 4; ++m) {
    if (m < nown) {
#pragma unroll
      for (int ks = 2 * m; ks < 2 * m + 2; ++ks) {
        const double a = ps[ks * 4 * LD];
        double b[4];
#pragma unroll
        for (int jj = 0; jj <= m; ++jj) b[jj] = ds[ks * 4 * (rho::NT + 4) + 8 * (J0 + jj)];
#pragma unroll
        for (int jj = 0; jj <= m; ++jj) dmma884(acc[J0 + jj][0], acc[J0 + jj][1], a, b[jj]);
      }
    }
  }
}

// TRI epilogue of the (up to 4) column groups J0.. that became final with this chunk: the Phi columns are the
// chunk's own first columns in the stage.  es points at column 2 r4, row 8 warp + q4 of the stage.
template <int J0>
__device__ __forceinline__ void rho_epi_smem(const double (&acc)[16][2], double& rs, const double* __restrict__ es,
                                             int ecnt) {
#pragma unroll
  for (int jj = 0; jj < 4; ++jj) {
    if (jj < ecnt) {
      const double* e = es + jj * 8 * LD;
      rs += acc[J0 + jj][0] * e[0] + acc[J0 + jj][1] * e[LD];
    }
  }
}

// GGA epilogue stage: column groups J0, J0+1 of the finished X tile against the staged Phi, dxPhi, dyPhi, dzPhi
// columns ([array][16 columns][LD]); es points at column 2 r4, row 8 warp + q4 of array 0.
// xg (optional): global X store of the nuclear-gradient path, at (column 2 r4 of this stage, row 8 warp + q4).
template <int J0>
__device__ __forceinline__ void rho_epi_gga(const double (&acc)[16][2], double (&rs)[4], const double* __restrict__ es,
                                            int eb, double* __restrict__ xg) {
#pragma unroll
  for (int jj = 0; jj < 2; ++jj) {
    if (jj < eb) {
      if (xg) {
        xg[(jj * 8) * GB] = acc[J0 + jj][0];
        xg[(jj * 8 + 1) * GB] = acc[J0 + jj][1];
      }
#pragma unroll
      for (int a = 0; a < 4; ++a) {
        const double* e = es + (a * rho::EC + jj * 8) * LD;
        rs[a] += acc[J0 + jj][0] * e[0] + acc[J0 + jj][1] * e[LD];
      }
    }
  }
}

// X-only epilogue (IMPL = 2, the X build of kldi_exc_grad): the stage holds 64 columns of Phi alone; column groups
// J0..J0+7 of the finished X tile give rho and go to the X store.  Four times fewer epilogue stages than the GGA form,
// and an epilogue stage costs one memory latency whatever it carries.
template <int J0>
__device__ __forceinline__ void rho_epi_x(const double (&acc)[16][2], double& rs, const double* __restrict__ es, int eb,
                                          double* __restrict__ xg) {
#pragma unroll
  for (int jj = 0; jj < 8; ++jj) {
    if (jj < eb) {
      const double* e = es + jj * 8 * LD;
      xg[(jj * 8) * GB] = acc[J0 + jj][0];
      xg[(jj * 8 + 1) * GB] = acc[J0 + jj][1];
      rs += acc[J0 + jj][0] * e[0] + acc[J0 + jj][1] * e[LD];
    }
  }
}

__device__ __forceinline__ void rho_stage(double (&acc)[16][2], const double* __restrict__ ps,
                                          const double* __restrict__ ds, int nks, int nj) {
  switch (nj) {
#define KLDI_CASE(N) case N: rho_ksteps<N>(acc, ps, ds, nks); break;
    KLDI_CASE(1) KLDI_CASE(2) KLDI_CASE(3) KLDI_CASE(4) KLDI_CASE(5) KLDI_CASE(6) KLDI_CASE(7) KLDI_CASE(8)
    KLDI_CASE(9) KLDI_CASE(10) KLDI_CASE(11) KLDI_CASE(12) KLDI_CASE(13) KLDI_CASE(14) KLDI_CASE(15) KLDI_CASE(16)
#undef KLDI_CASE
    default: break;
  }
}

// ------------------------------------------------------------------------------------ DFMA consumer (IMPL = 1)
// DMMA.8x8x4 tops out at 80 % of the FP64 unit rate on this part (profiles/r1f_summary.md); plain DFMA does not.  This
// consumer runs the LDA (triangular D') rho build on the vector pipe with register tiles.  8 consumer warps = 4 row
// blocks (wr) x 2 column halves (wc); a lane is (g = lane / 4, h = lane % 4): rows 32 wr + {2g, 2g+1, 16+2g, 17+2g},
// column owner o = 4 wc + h of the column PAIRS q = o, o+8, o+16, ... of the N-tile (columns 16 t + 2 o + {0,1}: cyclic,
// so that the triangular shape of D' loads every owner alike); tile width <= 64 -> 4 x 8 accumulators per lane (96 spills
// at the 170-register budget of 12 warps and ran slower).  Per k:
// two 16-byte loads of Phi (8 row groups x 16 B: one wavefront, broadcast over h) and one 16-byte load of D'[k][pair]
// per pair slot (4 owners x 16 B, broadcast over g), 8 DFMA per pair slot.  The producer side, the ring and the stage
// headers are those of the DMMA kernel.
namespace rho {
#ifndef KLDI_TW_F
#define KLDI_TW_F 64
#endif
constexpr int NCW_F = 8, TW_F = KLDI_TW_F, NTP_F = TW_F / 16;   // consumer warps, tile width, pair slots per owner
constexpr int RED_OFF = (SMEM_BYTES + 15) & ~15;         // [2 column halves][128 rows] partial row sums of a panel
constexpr int SMEM_BYTES_F = RED_OFF + 2 * GB * 8;
}  // namespace rho

__device__ __forceinline__ void rho_f_fma8(double (&acc)[4][2 * rho::NTP_F], int t, const double2& a01,
                                           const double2& a23, const double2& b) {
  acc[0][2 * t] = fma(a01.x, b.x, acc[0][2 * t]);
  acc[0][2 * t + 1] = fma(a01.x, b.y, acc[0][2 * t + 1]);
  acc[1][2 * t] = fma(a01.y, b.x, acc[1][2 * t]);
  acc[1][2 * t + 1] = fma(a01.y, b.y, acc[1][2 * t + 1]);
  acc[2][2 * t] = fma(a23.x, b.x, acc[2][2 * t]);
  acc[2][2 * t + 1] = fma(a23.x, b.y, acc[2][2 * t + 1]);
  acc[3][2 * t] = fma(a23.y, b.x, acc[3][2 * t]);
  acc[3][2 * t + 1] = fma(a23.y, b.y, acc[3][2 * t + 1]);
}

// Rectangle [0, cw) of the stage's columns: NTS pair slots of the warp's first owner; an owner whose last slot lies
// beyond cw multiplies zeros there (last_ok = 0).
template <int NTS>
__device__ __forceinline__ void rho_f_rect(double (&acc)[4][2 * rho::NTP_F], const double* __restrict__ pa,
                                           const double* __restrict__ db, int kc, bool last_ok) {
#pragma unroll 4
  for (int k = 0; k < kc; ++k) {
    const double2 a01 = *reinterpret_cast<const double2*>(pa + k * LD);
    const double2 a23 = *reinterpret_cast<const double2*>(pa + k * LD + 16);
#pragma unroll
    for (int t = 0; t < NTS; ++t) {
      if (t < rho::NTP_F) {
        double2 b = *reinterpret_cast<const double2*>(db + k * (rho::NT + 4) + 16 * t);
        if (t == NTS - 1 && !last_ok) b = make_double2(0.0, 0.0);
        rho_f_fma8(acc, t, a01, a23, b);
      }
    }
  }
}

// The chunk's own columns [o0, o0 + kc) of the tile (o0 = 16 T0): an owner's pairs there are slots T0 and T0 + 1,
// columns c = 16 t + 2 o.  D'[k][c] = 0 for chunk rows k < c - o0 (the stage holds those zeros), so every lane of the
// warp may start at the warp's first row 16 tt + 8 wc.  After the chunk these columns of X' are final and their Phi
// columns are the chunk's own columns c - o0 of the stage: epilogue.
template <int T0>
__device__ __forceinline__ void rho_f_diag(double (&acc)[4][2 * rho::NTP_F], double (&rs)[4],
                                           const double* __restrict__ pa, const double* __restrict__ db, int kc, int wc,
                                           int o) {
#pragma unroll
  for (int tt = 0; tt < 2; ++tt) {
    if (T0 + tt < rho::NTP_F) {
      const int k_lo = 16 * tt + 8 * wc;   // warp-uniform
      const int ks = 16 * tt + 2 * o;      // the lane's own first row = its pair's chunk column
      const bool valid = ks < kc;          // beyond a ragged last chunk the stage columns are not written
      if (k_lo < kc) {
        for (int k = k_lo; k < kc; ++k) {
          const double2 a01 = *reinterpret_cast<const double2*>(pa + k * LD);
          const double2 a23 = *reinterpret_cast<const double2*>(pa + k * LD + 16);
          double2 b = *reinterpret_cast<const double2*>(db + k * (rho::NT + 4) + 16 * (T0 + tt));
          if (!valid) b = make_double2(0.0, 0.0);
          rho_f_fma8(acc, T0 + tt, a01, a23, b);
        }
        if (valid) {
#pragma unroll
          for (int e = 0; e < 2; ++e) {  // epilogue: X'[rows][c + e] . Phi[rows][c + e], Phi column = chunk column ks + e
            const double2 p01 = *reinterpret_cast<const double2*>(pa + (ks + e) * LD);
            const double2 p23 = *reinterpret_cast<const double2*>(pa + (ks + e) * LD + 16);
            rs[0] = fma(acc[0][2 * (T0 + tt) + e], p01.x, rs[0]);
            rs[1] = fma(acc[1][2 * (T0 + tt) + e], p01.y, rs[1]);
            rs[2] = fma(acc[2][2 * (T0 + tt) + e], p23.x, rs[2]);
            rs[3] = fma(acc[3][2 * (T0 + tt) + e], p23.y, rs[3]);
          }
        }
      }
    }
  }
}

__device__ __forceinline__ void rho_consumer_dfma(unsigned char* smem, const int* hdr, uint32_t bar0,
                                                  double* __restrict__ rho_s, int warp, int lane) {
  using namespace rho;
  double acc[4][2 * NTP_F];
  double rs[4] = {0.0, 0.0, 0.0, 0.0};
  double* red = reinterpret_cast<double*>(smem + RED_OFF);
  const int wr = warp >> 1, wc = warp & 1, g = lane >> 2, h = lane & 3, o = 4 * wc + h;
  int s = 0;
  uint32_t ph = 0;
  for (;;) {
    mbar_wait(bar0 + 8 * s, ph);
    const int p = hdr[4 * s + 0], h2 = hdr[4 * s + 2], h3 = hdr[4 * s + 3];
    const int fl = h2 >> 16;
    if (fl & F_DONE) break;
    const int kc = (h2 & 0xff) * 4, wact = ((h2 >> 8) & 0xff) * 8, ecnt = h3 >> 16, o0 = ((h3 >> 8) & 0xff) * 8;
    if (fl & F_FIRST) {
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 2 * NTP_F; ++j) acc[i][j] = 0.0;
    }
    const double* pa = reinterpret_cast<const double*>(smem + s * STAGE_BYTES) + 32 * wr + 2 * g;   // rows of column k
    const double* db = reinterpret_cast<const double*>(smem + s * STAGE_BYTES + PHI_BYTES) + 2 * o;  // pair slot 0
    const int cw = ecnt ? o0 : wact;                                   // width of the rectangle before the own columns
    const int nts = cw > 8 * wc ? (cw - 8 * wc + 15) >> 4 : 0;         // pair slots of the warp's first owner (uniform)
    const bool last_ok = 16 * (nts - 1) + 2 * o < cw;                  // this lane's last slot is inside the rectangle
    switch (nts) {
      case 1: rho_f_rect<1>(acc, pa, db, kc, last_ok); break;
      case 2: rho_f_rect<2>(acc, pa, db, kc, last_ok); break;
      case 3: rho_f_rect<3>(acc, pa, db, kc, last_ok); break;
      case 4: rho_f_rect<4>(acc, pa, db, kc, last_ok); break;
      case 5: rho_f_rect<5>(acc, pa, db, kc, last_ok); break;
      case 6: rho_f_rect<6>(acc, pa, db, kc, last_ok); break;
      default: break;
    }
    if (ecnt) {
      switch (o0 >> 5) {
        case 0: rho_f_diag<0>(acc, rs, pa, db, kc, wc, o); break;
        case 1: rho_f_diag<2>(acc, rs, pa, db, kc, wc, o); break;
        default: rho_f_diag<4>(acc, rs, pa, db, kc, wc, o); break;
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(bar0 + 8 * (NST + s));
    if (++s == NST) { s = 0; ph ^= 1; }

    if (fl & F_LAST_PANEL) {  // rho_p: the 4 owners of a warp by shuffle, the 2 column halves through shared memory
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        rs[i] += __shfl_xor_sync(0xffffffffu, rs[i], 1);
        rs[i] += __shfl_xor_sync(0xffffffffu, rs[i], 2);
      }
      if (h == 0) {
        *reinterpret_cast<double2*>(red + wc * GB + 32 * wr + 2 * g) = make_double2(rs[0], rs[1]);
        *reinterpret_cast<double2*>(red + wc * GB + 32 * wr + 16 + 2 * g) = make_double2(rs[2], rs[3]);
      }
      rs[0] = rs[1] = rs[2] = rs[3] = 0.0;
      asm volatile("bar.sync 2, %0;" ::"n"(32 * NCW_F) : "memory");
      const int r = warp * 32 + lane;
      if (r < GB) rho_s[(int64_t)p * GB + r] = 2.0 * (red[r] + red[GB + r]);
      asm volatile("bar.sync 2, %0;" ::"n"(32 * NCW_F) : "memory");
    }
  }
}

template <bool GGA, bool TRI, int IMPL = 0>
__global__ void __launch_bounds__(IMPL == 1 ? 32 * (rho::NCW_F + rho::NPW) : rho::NTHREADS, 1)
    k_rho(const int32_t* __restrict__ tasks, int n_tasks, int32_t* __restrict__ ticket,
          const int32_t* __restrict__ kp, const int64_t* __restrict__ panel_off, const int32_t* __restrict__ colidx,
          const double* __restrict__ phi, const double* __restrict__ dphi0, const double* __restrict__ dphi1,
          const double* __restrict__ dphi2, const double* __restrict__ Dp, int n_ao, double* __restrict__ rho_s,
          double* __restrict__ drho_s, int64_t n_pad, const unsigned long long* __restrict__ pmask,
          double* __restrict__ x_store) {
  using namespace rho;
  static_assert(IMPL != 1 || (TRI && !GGA), "the DFMA consumer implements the LDA (triangular) form");
  static_assert(IMPL != 2 || (GGA && !TRI), "the X-only epilogue belongs to the full-D form");
  constexpr int NCWI = IMPL == 1 ? NCW_F : NCW;  // consumer warps
  constexpr int TW = IMPL == 1 ? TW_F : NT;      // N-tile width
  constexpr int ECI = IMPL == 2 ? 64 : EC;       // tile columns per epilogue stage
  extern __shared__ __align__(128) unsigned char smem[];
  int* hdr = reinterpret_cast<int*>(smem + NST * STAGE_BYTES);
  const uint32_t bar0 = smem_u32(smem + NST * STAGE_BYTES + NST * 16);  // full[s] at +8s, empty[s] at +8(NST+s)
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid == 0) {
    for (int s = 0; s < NST; ++s) {
      mbar_init(bar0 + 8 * s, 1 + 32 * NPW);  // expect_tx arrive + one cp.async completion per producer lane
      mbar_init(bar0 + 8 * (NST + s), NCWI);  // one arrive per consumer warp
    }
    fence_mbar_init();
  }
  __syncthreads();

  if (warp >= NCWI) {
    // ------------------------------------------------------------------ producer warps (in lockstep per task)
    const int pw = warp - NCWI;
    volatile int* task_slot = reinterpret_cast<volatile int*>(smem + NST * STAGE_BYTES + NST * 16 + 2 * NST * 8);
    int s = 0;
    uint32_t ph = 0;
    for (;;) {
      if (pw == 0 && lane == 0) *task_slot = atomicAdd(ticket, 1);
      asm volatile("bar.sync 1, %0;" ::"n"(32 * NPW) : "memory");
      const int t = *task_slot;
      asm volatile("bar.sync 1, %0;" ::"n"(32 * NPW) : "memory");
      if (t >= n_tasks) break;
      const int p = tasks[t];
      const int K8 = (kp[p] + 7) & ~7;
      const int64_t base = panel_off[p];
      const int ntile = (K8 + TW - 1) / TW;
      // executable-pair mask of this grid block (pairsel.cu; Eq. 19): bit (k0/32)*4 + jt, all ones = no test
      const unsigned long long pm = pmask ? pmask[p] : ~0ull;
      // TRI: tiles start on 32-column (K-chunk) boundaries so that a chunk's own columns are whole j-groups
      const int W = TRI ? (((K8 + ntile - 1) / ntile) + 31) & ~31 : (((K8 + ntile - 1) / ntile) + 7) & ~7;
      for (int jt = 0; jt < ntile; ++jt) {
        const int n0 = jt * W, Wj = min(W, K8 - n0);
        int cn[4];
#pragma unroll
        for (int c = 0; c < 4; ++c) cn[c] = (lane + 32 * c < Wj) ? colidx[base + n0 + lane + 32 * c] : -1;
        // TRI: D' is lower triangular in packed order (colidx ascends), so chunk rows k < n0 contribute
        // nothing to this N-tile and a chunk [k0, k0+kc) only reaches the columns n < k0 + kc.
        // TRI also walks the chunks in DESCENDING k: after chunk [k0, k0+kc) the columns n in that same range of
        // X' = Phi D' are final (they only take k >= n) while their Phi columns are still in the stage, so the
        // rho epilogue of those columns runs from shared memory, chunk by chunk, with no global re-read.
        const int kstart = TRI ? n0 : 0;
        const int nchunk = (K8 - kstart + KC - 1) / KC;
        bool started = false;
        for (int ci = 0; ci < nchunk; ++ci) {
          const int k0 = kstart + KC * (TRI ? nchunk - 1 - ci : ci);
          const int kc = min(KC, K8 - k0);
          // a stage without an executable pair is skipped; the chunks that carry the tile's own columns (TRI:
          // their epilogue runs in that stage) and the last stage of a tile (it closes the tile) always run
          if (pm != ~0ull && !((pm >> (((k0 >> 5) & 15) * 4 + (jt & 3))) & 1ull) &&
              (TRI ? k0 >= n0 + Wj : ci != nchunk - 1))
            continue;
          const int wact = TRI ? min(Wj, k0 + kc - n0) : Wj;
          mbar_wait(bar0 + 8 * (NST + s), ph ^ 1);
          const int r0 = 8 * pw, r1 = min(kc, r0 + 8);  // this warp's rows of the chunk
          const int rowidx = (r0 + lane < r1) ? colidx[base + k0 + r0 + lane] : 0;
          const uint32_t full = bar0 + 8 * s;
          if (pw == 0 && lane == 0) {
            int fl = 0;
            if (!started) fl |= F_FIRST;
            if (ci == nchunk - 1) {
              if (!GGA) {
                fl |= F_LAST_TILE;
                if (jt == ntile - 1) fl |= F_LAST_PANEL;
              }
            }
            hdr[4 * s + 0] = p;
            hdr[4 * s + 1] = n0;
            hdr[4 * s + 2] = (kc >> 2) | ((wact >> 3) << 8) | (fl << 16);
            const int ecnt = TRI ? max(0, min(kc, n0 + Wj - k0)) >> 3 : 0;  // final column groups of this chunk
            hdr[4 * s + 3] = (Wj >> 3) | (((k0 - n0) >> 3) << 8) | (ecnt << 16);
            mbar_arrive_expect_tx(full, (uint32_t)kc * (GB * 8));
          }
          __syncwarp();
          const uint32_t sphi = smem_u32(smem + s * STAGE_BYTES);
          const uint32_t sd = sphi + PHI_BYTES;
          if (r0 + lane < r1)
            bulk_g2s(sphi + (r0 + lane) * (LD * 8), phi + (base + k0 + r0 + lane) * GB, GB * 8, full);
          for (int r = r0; r < r1; ++r) {
            const int row = __shfl_sync(0xffffffffu, rowidx, r - r0);
            const double* drow = Dp + (int64_t)row * n_ao;
            const uint32_t dst = sd + (r * (NT + 4) + lane) * 8;
#pragma unroll
            for (int c = 0; c < 4; ++c)
              if (cn[c] >= 0 && lane + 32 * c < wact) cp_async8(dst + c * 256, drow + cn[c]);
          }
          cp_async_mbar_arrive_noinc(full);
          started = true;
          if (++s == NST) { s = 0; ph ^= 1; }
        }
        if (GGA) {
          // epilogue operands through the ring: stage e holds columns [n0+16e, n0+16e+16) of the four stores,
          // producer warp a stages array a; the consumers contract them with the finished X tile from shared memory
          const double* arr = pw == 0 ? phi : pw == 1 ? dphi0 : pw == 2 ? dphi1 : dphi2;
          const int nes = (Wj + ECI - 1) / ECI;
          for (int e = 0; e < nes; ++e) {
            const int ec = min(ECI, Wj - ECI * e);
            mbar_wait(bar0 + 8 * (NST + s), ph ^ 1);
            const uint32_t full = bar0 + 8 * s;
            if (pw == 0 && lane == 0) {
              hdr[4 * s + 0] = p;
              hdr[4 * s + 1] = n0;
              hdr[4 * s + 2] = (F_EPI | ((e == nes - 1 && jt == ntile - 1) ? F_LAST_PANEL : 0)) << 16;
              hdr[4 * s + 3] = e | ((ec >> 3) << 8);
              mbar_arrive_expect_tx(full, (uint32_t)((IMPL == 2 ? 1 : 4) * ec) * (GB * 8));
            }
            __syncwarp();
            if (IMPL == 2) {  // Phi alone, 64 columns: producer warp pw copies columns 16 pw .. 16 pw + 15
              if (lane < 16 && 16 * pw + lane < ec)
                bulk_g2s(smem_u32(smem + s * STAGE_BYTES) + (16 * pw + lane) * (LD * 8),
                         phi + (base + n0 + ECI * e + 16 * pw + lane) * GB, GB * 8, full);
            } else if (lane < ec)
              bulk_g2s(smem_u32(smem + s * STAGE_BYTES) + (pw * EC + lane) * (LD * 8),
                       arr + (base + n0 + EC * e + lane) * GB, GB * 8, full);
            cp_async_mbar_arrive_noinc(full);
            if (++s == NST) { s = 0; ph ^= 1; }
          }
        }
      }
    }
    mbar_wait(bar0 + 8 * (NST + s), ph ^ 1);
    if (pw == 0 && lane == 0) {
      hdr[4 * s + 2] = F_DONE << 16;
      mbar_arrive(bar0 + 8 * s);
    }
    cp_async_mbar_arrive_noinc(bar0 + 8 * s);
    return;
  }

  if constexpr (IMPL == 1) {
    rho_consumer_dfma(smem, hdr, bar0, rho_s, warp, lane);
    return;
  }
  // -------------------------------------------------------------------- consumer warps (8 rows each)
  double acc[16][2];
  double rs[GGA ? 4 : 1];
#pragma unroll
  for (int c = 0; c < (GGA ? 4 : 1); ++c) rs[c] = 0.0;
  int s = 0;
  uint32_t ph = 0;
  const int q4 = lane >> 2, r4 = lane & 3;
  for (;;) {
    mbar_wait(bar0 + 8 * s, ph);
    const int p = hdr[4 * s + 0], h2 = hdr[4 * s + 2];
    const int fl = h2 >> 16;
    if (fl & F_DONE) break;
    const int nks = h2 & 0xff, nj = (h2 >> 8) & 0xff, h3 = hdr[4 * s + 3];
    const double* es = reinterpret_cast<const double*>(smem + s * STAGE_BYTES) + 2 * r4 * LD + 8 * warp + q4;
    if (GGA && (fl & F_EPI)) {
      if constexpr (GGA) {
        const int eb = h3 >> 8;  // 8-column groups in this stage (1 or 2; X-only form: up to 8)
        double* xg = nullptr;
        if (x_store)
          xg = x_store + (panel_off[p] + hdr[4 * s + 1] + ECI * (h3 & 0xff) + 2 * r4) * GB + 8 * warp + q4;
        if constexpr (IMPL == 2) {
          if ((h3 & 0xff) == 0)
            rho_epi_x<0>(acc, rs[0], es, eb, xg);
          else
            rho_epi_x<8>(acc, rs[0], es, eb, xg);
        } else
        switch (h3 & 0xff) {
#define KLDI_CASE(E) case E: rho_epi_gga<2 * E>(acc, rs, es, eb, xg); break;
          KLDI_CASE(0) KLDI_CASE(1) KLDI_CASE(2) KLDI_CASE(3) KLDI_CASE(4) KLDI_CASE(5) KLDI_CASE(6) KLDI_CASE(7)
#undef KLDI_CASE
          default: break;
        }
      }
    } else {
      if (fl & F_FIRST) {
#pragma unroll
        for (int j = 0; j < 16; ++j) acc[j][0] = acc[j][1] = 0.0;
      }
      const double* ps = reinterpret_cast<const double*>(smem + s * STAGE_BYTES) + r4 * LD + 8 * warp + q4;
      const double* ds = reinterpret_cast<const double*>(smem + s * STAGE_BYTES + PHI_BYTES) + r4 * (NT + 4) + q4;
      const int ecnt = TRI ? h3 >> 16 : 0;
      if (TRI && ecnt) {
        // diagonal chunk: rectangle of the columns before the chunk's own, then the triangular own block
        rho_stage(acc, ps, ds, nks, (h3 >> 8) & 0xff);
        switch ((h3 >> 10) & 3) {  // first own (= final) column group / 4
#define KLDI_CASE(Q) \
  case Q: rho_diag<4 * Q>(acc, ps, ds, ecnt); rho_epi_smem<4 * Q>(acc, rs[0], es, ecnt); break;
          KLDI_CASE(0) KLDI_CASE(1) KLDI_CASE(2)
#undef KLDI_CASE
          default: rho_diag<12>(acc, ps, ds, ecnt); rho_epi_smem<12>(acc, rs[0], es, ecnt); break;
        }
      } else {
        rho_stage(acc, ps, ds, nks, nj);
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(bar0 + 8 * (NST + s));
    if (++s == NST) { s = 0; ph ^= 1; }

    if (fl & F_LAST_PANEL) {  // rho_p (and grad rho_p) of this warp's 8 rows: quad reduction, one store per row
#pragma unroll
      for (int c = 0; c < ((GGA && IMPL != 2) ? 4 : 1); ++c) {
        double v = rs[c];
        v += __shfl_xor_sync(0xffffffffu, v, 1);
        v += __shfl_xor_sync(0xffffffffu, v, 2);
        if (r4 == 0) {
          const int64_t g = (int64_t)p * GB + 8 * warp + q4;
          if (c == 0)
            rho_s[g] = TRI ? 2.0 * v : v;
          else
            drho_s[(int64_t)(c - 1) * n_pad + g] = 2.0 * v;
        }
        rs[c] = 0.0;
      }
    }
  }
}

static kldi_status set_attrs(const kldi_plan* P);

// ===================================================================================== H3
constexpr double C_X = 0.73855876638202240588;    // (3/4)(3/pi)^{1/3}
constexpr double K_S = 9.5707800006273016908;     // (3 pi^2)^{2/3}
constexpr double PBE_KAPPA = 0.804, PBE_MU = 0.21951, RHO_CUT = 1e-20;

template <bool GGA>
__global__ void __launch_bounds__(256) k_xc(int64_t n_pad, const double* __restrict__ rho_s,
                                            const double* __restrict__ drho_s, const double* __restrict__ gw,
                                            double* __restrict__ wv_s, double* __restrict__ epart) {
  __shared__ double red[256];
  const int64_t g = (int64_t)blockIdx.x * 256 + threadIdx.x;
  double we = 0.0;
  if (g < n_pad) {
    const double r = rho_s[g], w = gw[g];
    double v0 = 0.0, v1 = 0.0, v2 = 0.0, v3 = 0.0;
    if (r >= RHO_CUT) {
      const double c = cbrt(r);
      if (!GGA) {
        we = w * (-C_X * r * c);
        v0 = w * (-(4.0 / 3.0) * C_X * c);
      } else {
        const double dx = drho_s[g], dy = drho_s[n_pad + g], dz = drho_s[2 * n_pad + g];
        const double sigma = dx * dx + dy * dy + dz * dz;
        const double r43 = r * c;
        const double s2 = sigma / (4.0 * K_S * r43 * r43);
        const double den = 1.0 + PBE_MU * s2 / PBE_KAPPA;
        const double F = 1.0 + PBE_KAPPA - PBE_KAPPA / den;
        const double Fp = PBE_MU / (den * den);
        we = w * (-C_X * r43 * F);
        v0 = w * (-C_X * c * ((4.0 / 3.0) * F - (8.0 / 3.0) * s2 * Fp));
        const double vs = -C_X * Fp / (4.0 * K_S * r43);
        v1 = 2.0 * w * vs * dx;
        v2 = 2.0 * w * vs * dy;
        v3 = 2.0 * w * vs * dz;
      }
    }
    wv_s[g] = v0;
    if (GGA) {
      wv_s[n_pad + g] = v1;
      wv_s[2 * n_pad + g] = v2;
      wv_s[3 * n_pad + g] = v3;
    }
  }
  red[threadIdx.x] = we;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {  // fixed tree: bitwise reproducible
    if (threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
    __syncthreads();
  }
  if (threadIdx.x == 0) epart[blockIdx.x] = red[0];
}

__global__ void __launch_bounds__(1024) k_sum_partials(const double* __restrict__ part, int n, double* __restrict__ out) {
  __shared__ double red[1024];
  double a = 0.0;
  for (int i = threadIdx.x; i < n; i += 1024) a += part[i];
  red[threadIdx.x] = a;
  __syncthreads();
  for (int o = 512; o > 0; o >>= 1) {
    if (threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
    __syncthreads();
  }
  if (threadIdx.x == 0) out[0] = red[0];
}

// ===================================================================================== nuclear gradient
// dE_xc/dA_c = -2 sum_g wv_g sum_{mu on A} d_c Phi_{g,mu} X_{g,mu} (LDA, fixed grid, G1):
// one CTA per grid block, one warp per retained column; X comes from the store the rho kernel wrote.  HBM-bound
// (X and the three gradient stores are read once).
__global__ void __launch_bounds__(256) k_grad_cols(const int32_t* __restrict__ tasks, const int32_t* __restrict__ kp,
                                                   const int64_t* __restrict__ panel_off,
                                                   const int32_t* __restrict__ colidx,
                                                   const int32_t* __restrict__ ao_atom_c, const double* __restrict__ x,
                                                   const double* __restrict__ d0, const double* __restrict__ d1,
                                                   const double* __restrict__ d2, const double* __restrict__ wv_s,
                                                   double* __restrict__ grad) {
  const int p = tasks[blockIdx.x], lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int K = kp[p];
  const int64_t base = panel_off[p];
  double w[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) w[i] = wv_s[(int64_t)p * GB + 4 * lane + i];
  for (int k = warp; k < K; k += 8) {
    const int64_t o = (base + k) * GB + 4 * lane;
    double t[3] = {0.0, 0.0, 0.0};
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const double2 xv = *reinterpret_cast<const double2*>(x + o + 2 * h);
      const double2 a = *reinterpret_cast<const double2*>(d0 + o + 2 * h);
      const double2 b = *reinterpret_cast<const double2*>(d1 + o + 2 * h);
      const double2 c = *reinterpret_cast<const double2*>(d2 + o + 2 * h);
      const double x0 = w[2 * h] * xv.x, x1 = w[2 * h + 1] * xv.y;
      t[0] += x0 * a.x + x1 * a.y;
      t[1] += x0 * b.x + x1 * b.y;
      t[2] += x0 * c.x + x1 * c.y;
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) {
#pragma unroll
      for (int m = 16; m > 0; m >>= 1) t[c] += __shfl_xor_sync(0xffffffffu, t[c], m);
    }
    if (lane < 3) {
      const int atom = ao_atom_c[colidx[base + k]];
      atomicAdd(grad + 3 * atom + lane, -2.0 * (lane == 0 ? t[0] : lane == 1 ? t[1] : t[2]));
    }
  }
}

// GGA form (G1):
//   dE/dA_c = -2 sum_g sum_{mu on A} { wv0 d_c Phi_mu X_mu + sum_d wv_d [ d_c d_d Phi_mu X_mu + d_c Phi_mu X^d_mu ] },
// wv0 = w v_rho, wv_d = 2 w v_sigma d_d rho (k_xc), X = Phi D and X^d = d_d Phi D from the stores the rho kernel wrote.
// One CTA per grid block, one thread per grid point; the first and second AO derivatives of a column are evaluated
// from the shell table (no Hessian store); the columns of a panel ascend in plan AO index, so an atom's columns are
// consecutive: the three components are summed over them in registers and reduced over the block once per atom.
__global__ void __launch_bounds__(128) k_grad_cols_gga(ShellTable T, const int32_t* __restrict__ tasks,
                                                       const int32_t* __restrict__ kp, const int64_t* __restrict__ panel_off,
                                                       const int32_t* __restrict__ colidx, const int32_t* __restrict__ ao_shell,
                                                       const int32_t* __restrict__ ao_atom_c, const double* __restrict__ gx,
                                                       const double* __restrict__ gy, const double* __restrict__ gz,
                                                       const double* __restrict__ x, const double* __restrict__ xd,
                                                       int64_t xd_stride, const double* __restrict__ wv_s, int64_t n_pad,
                                                       double* __restrict__ grad) {
  __shared__ double red[4][3];
  const int p = tasks[blockIdx.x], t = threadIdx.x, lane = t & 31, warp = t >> 5;
  const int K = kp[p];
  const int64_t base = panel_off[p], g = (int64_t)p * GB + t;
  const double px = gx[g], py = gy[g], pz = gz[g];
  const double w0 = wv_s[g], w1 = wv_s[n_pad + g], w2 = wv_s[2 * n_pad + g], w3 = wv_s[3 * n_pad + g];
  double acc[3] = {0.0, 0.0, 0.0};
  int cur_atom = -1;
  auto flush = [&](int atom) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      double v = acc[c];
#pragma unroll
      for (int m = 16; m > 0; m >>= 1) v += __shfl_xor_sync(0xffffffffu, v, m);
      if (lane == 0) red[warp][c] = v;
      acc[c] = 0.0;
    }
    __syncthreads();
    if (t < 3) atomicAdd(grad + 3 * atom + t, -2.0 * (red[0][t] + red[1][t] + red[2][t] + red[3][t]));
    __syncthreads();
  };
  for (int k = 0; k < K; ++k) {
    const int ao = colidx[base + k];
    const int atom = ao_atom_c[ao];
    if (atom != cur_atom) {
      if (cur_atom >= 0) flush(cur_atom);
      cur_atom = atom;
    }
    const int s = ao_shell[ao];
    double gr[3], h[6];
    eval_component_hess(T, s, ao - T.sh_ao0[s], px, py, pz, gr, h);
    const int64_t o = (base + k) * GB + t;
    const double X = x[o], X0 = xd[o], X1 = xd[xd_stride + o], X2 = xd[2 * xd_stride + o];
    const double xw = w0 * X + w1 * X0 + w2 * X1 + w3 * X2;  // multiplies d_c Phi
    acc[0] += gr[0] * xw + X * (w1 * h[0] + w2 * h[1] + w3 * h[2]);
    acc[1] += gr[1] * xw + X * (w1 * h[1] + w2 * h[3] + w3 * h[4]);
    acc[2] += gr[2] * xw + X * (w1 * h[2] + w2 * h[4] + w3 * h[5]);
  }
  if (cur_atom >= 0) flush(cur_atom);
}

kldi_status launch_grad_cols(kldi_plan* P, double* grad) {
  KLDI_CUDA(cudaMemsetAsync(grad, 0, sizeof(double) * 3 * P->n_atoms, P->stream));
  if (P->n_tasks == 0) return KLDI_OK;
  k_grad_cols<<<P->n_tasks, 256, 0, P->stream>>>(P->d_tasks, P->d_kp, P->d_panel_off, P->d_colidx, P->d_ao_atom_c,
                                                 P->d_x, P->d_dphi[0], P->d_dphi[1], P->d_dphi[2], P->d_wv_s, grad);
  KLDI_LAUNCHED(P);
  return KLDI_OK;
}

kldi_status launch_grad_cols_gga(kldi_plan* P, double* grad) {
  KLDI_CUDA(cudaMemsetAsync(grad, 0, sizeof(double) * 3 * P->n_atoms, P->stream));
  if (P->n_tasks == 0) return KLDI_OK;
  ShellTable T{P->d_atom_xyz, P->d_sh_atom, P->d_sh_l, P->d_sh_prim0, P->d_sh_ao0, P->d_prim_alpha, P->d_prim_cn};
  const int64_t stride = (int64_t)GB * (P->total_cols + 64);
  k_grad_cols_gga<<<P->n_tasks, 128, 0, P->stream>>>(T, P->d_tasks, P->d_kp, P->d_panel_off, P->d_colidx, P->d_ao_shell,
                                                     P->d_ao_atom_c, P->d_gx, P->d_gy, P->d_gz, P->d_x, P->d_xd, stride,
                                                     P->d_wv_s, P->n_pad, grad);
  KLDI_LAUNCHED(P);
  return KLDI_OK;
}

// X_out = A D for another store A of the rho layout (A = d_d Phi: the X^d of the GGA nuclear gradient), with the X-only
// form of k_rho; its row sums go to a scratch vector.  The full D must already be in P->d_Dp.
kldi_status launch_x_on(kldi_plan* P, const double* store, double* x_out, double* rho_scratch) {
  kldi_status rc = set_attrs(P);
  if (rc != KLDI_OK) return rc;
  KLDI_CUDA(cudaMemsetAsync(P->d_ticket, 0, sizeof(int32_t) * 4, P->stream));
  if (P->n_tasks == 0) return KLDI_OK;
  const int grid = P->n_sm < P->n_tasks ? P->n_sm : P->n_tasks;
  k_rho<true, false, 2><<<grid, rho::NTHREADS, rho::SMEM_BYTES, P->stream>>>(
      P->d_tasks, P->n_tasks, P->d_ticket, P->d_kp, P->d_panel_off, P->d_colidx, store, nullptr, nullptr, nullptr, P->d_Dp,
      P->n_ao, rho_scratch, nullptr, P->n_pad, nullptr, x_out);
  KLDI_LAUNCHED(P);
  return KLDI_OK;
}

// ===================================================================================== permutations
__global__ void k_unpermute_rho(const int32_t* __restrict__ perm, int64_t n_pad, int64_t n_pts,
                                const double* __restrict__ rho_s, const double* __restrict__ drho_s,
                                double* __restrict__ rho, double* __restrict__ drho) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_pad) return;
  const int64_t g = perm[i];
  if (g < 0) return;
  rho[g] = rho_s[i];
  if (drho)
    for (int c = 0; c < 3; ++c) drho[c * n_pts + g] = drho_s[c * n_pad + i];
}

__global__ void k_gather_wv(const int32_t* __restrict__ perm, int64_t n_pad, int64_t n_pts, int ncomp,
                            const double* __restrict__ wv, double* __restrict__ wv_s, double scale) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_pad) return;
  const int64_t g = perm[i];
  for (int c = 0; c < ncomp; ++c) wv_s[c * n_pad + i] = (g >= 0) ? scale * wv[c * n_pts + g] : 0.0;
}

// tau_g = 1/2 sum_c t_c(g), t_c = sum_{mu,nu} D_{mu,nu} d_c chi_mu d_c chi_nu from three LDA-form rho builds
__global__ void k_tau_combine(int64_t n_pad, const double* __restrict__ t, double* __restrict__ tau_s) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n_pad) tau_s[i] = 0.5 * (t[i] + t[n_pad + i] + t[2 * n_pad + i]);
}

// H4 (V contraction) lives in vgram.cu.

// ===================================================================================== H5
// FIXED: Vp holds 64-bit fixed-point sums (k_vgram EPI = 2); back to double with the exact power-of-two scale.
template <bool GGA, bool FIXED>
__global__ void k_finalise_V(const double* __restrict__ Vp, const int32_t* __restrict__ ao_perm, int n,
                             double* __restrict__ V, const double* __restrict__ fx_bound) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x, i = blockIdx.y;
  if (j >= n) return;
  const double inv = FIXED ? 1.0 / fx_scale(*fx_bound) : 1.0;
  auto ld = [&](int64_t o) {
    return FIXED ? (double)__double_as_longlong(Vp[o]) * inv : Vp[o];
  };
  double v;
  if (GGA)
    v = ld((int64_t)i * n + j) + ld((int64_t)j * n + i);  // V = B + B^T (commutative: exactly symmetric)
  else
    v = (i <= j) ? ld((int64_t)i * n + j) : ld((int64_t)j * n + i);
  V[(int64_t)ao_perm[i] * n + ao_perm[j]] = v;
}

// ===================================================================================== launchers
static kldi_status set_attrs(const kldi_plan* P) {
  kldi_status rc;
  if ((rc = ensure_smem_attr((const void*)k_rho<false, true>, rho::SMEM_BYTES, P->device)) != KLDI_OK) return rc;
  if ((rc = ensure_smem_attr((const void*)k_rho<true, false>, rho::SMEM_BYTES, P->device)) != KLDI_OK) return rc;
  if ((rc = ensure_smem_attr((const void*)k_rho<false, true, 1>, rho::SMEM_BYTES_F, P->device)) != KLDI_OK) return rc;
  return ensure_smem_attr((const void*)k_rho<true, false, 2>, rho::SMEM_BYTES, P->device);
}

kldi_status launch_permute_D(kldi_plan* P, const double* D, bool gga) {
  dim3 grid((P->n_ao + 255) / 256, P->n_ao);
  if (gga)  // the GGA epilogue needs the full X = Phi D for grad rho; LDA uses the triangular form
    k_permute_D<false><<<grid, 256, 0, P->stream>>>(D, P->d_ao_perm, P->n_ao, P->d_Dp);
  else
    k_permute_D<true><<<grid, 256, 0, P->stream>>>(D, P->d_ao_perm, P->n_ao, P->d_Dp);
  KLDI_LAUNCHED(P);
  return KLDI_OK;
}

kldi_status launch_rho(kldi_plan* P, bool gga, double* x_store, bool x_only) {
  kldi_status rc = set_attrs(P);
  if (rc != KLDI_OK) return rc;
  if (!gga && P->rho_impl == 2 && !P->pair_test) return launch_rho_tc(P);
  KLDI_CUDA(cudaMemsetAsync(P->d_rho_s, 0, sizeof(double) * P->n_pad, P->stream));
  if (gga) KLDI_CUDA(cudaMemsetAsync(P->d_drho_s, 0, sizeof(double) * 3 * P->n_pad, P->stream));
  KLDI_CUDA(cudaMemsetAsync(P->d_ticket, 0, sizeof(int32_t) * 4, P->stream));
  if (P->n_tasks == 0) return KLDI_OK;
  const unsigned long long* pm = nullptr;
  if (P->pair_test) {
    if ((rc = launch_pair_select(P, !gga)) != KLDI_OK) return rc;
    pm = P->d_pmask;
  }
  const int grid = P->n_sm < P->n_tasks ? P->n_sm : P->n_tasks;
  if (gga && x_store && x_only)  // the X build of kldi_exc_grad (LDA): rho and the X store, no grad rho
    k_rho<true, false, 2><<<grid, rho::NTHREADS, rho::SMEM_BYTES, P->stream>>>(
        P->d_tasks, P->n_tasks, P->d_ticket, P->d_kp, P->d_panel_off, P->d_colidx, P->d_phi, nullptr, nullptr, nullptr,
        P->d_Dp, P->n_ao, P->d_rho_s, P->d_drho_s, P->n_pad, pm, x_store);
  else if (gga)
    k_rho<true, false><<<grid, rho::NTHREADS, rho::SMEM_BYTES, P->stream>>>(P->d_tasks, P->n_tasks, P->d_ticket, P->d_kp, P->d_panel_off,
                                                           P->d_colidx, P->d_phi, P->d_dphi[0], P->d_dphi[1],
                                                           P->d_dphi[2], P->d_Dp, P->n_ao, P->d_rho_s, P->d_drho_s,
                                                           P->n_pad, pm, x_store);
  else if (P->rho_impl == 1 && !pm)
    k_rho<false, true, 1><<<grid, 32 * (rho::NCW_F + rho::NPW), rho::SMEM_BYTES_F, P->stream>>>(
        P->d_tasks, P->n_tasks, P->d_ticket, P->d_kp, P->d_panel_off, P->d_colidx, P->d_phi, nullptr, nullptr, nullptr,
        P->d_Dp, P->n_ao, P->d_rho_s, nullptr, P->n_pad, nullptr, nullptr);
  else
    k_rho<false, true><<<grid, rho::NTHREADS, rho::SMEM_BYTES, P->stream>>>(P->d_tasks, P->n_tasks, P->d_ticket, P->d_kp,
                                                            P->d_panel_off, P->d_colidx, P->d_phi, nullptr, nullptr,
                                                            nullptr, P->d_Dp, P->n_ao, P->d_rho_s, nullptr, P->n_pad,
                                                            pm, nullptr);
  KLDI_LAUNCHED(P);
  return KLDI_OK;
}

// The LDA-form (triangular D') rho build on another store of the rho layout: out_s[g] = sum_{mu,nu} D_{mu,nu}
// A_{g,mu} A_{g,nu} with A = d_c Phi (kinetic-energy density).  D' must already be in P->d_Dp.
kldi_status launch_rho_lda_on(kldi_plan* P, const double* store, double* out_s) {
  kldi_status rc = set_attrs(P);
  if (rc != KLDI_OK) return rc;
  KLDI_CUDA(cudaMemsetAsync(out_s, 0, sizeof(double) * P->n_pad, P->stream));
  KLDI_CUDA(cudaMemsetAsync(P->d_ticket, 0, sizeof(int32_t) * 4, P->stream));
  if (P->n_tasks == 0) return KLDI_OK;
  const int grid = P->n_sm < P->n_tasks ? P->n_sm : P->n_tasks;
  k_rho<false, true><<<grid, rho::NTHREADS, rho::SMEM_BYTES, P->stream>>>(
      P->d_tasks, P->n_tasks, P->d_ticket, P->d_kp, P->d_panel_off, P->d_colidx, store, nullptr, nullptr, nullptr,
      P->d_Dp, P->n_ao, out_s, nullptr, P->n_pad, nullptr, nullptr);
  KLDI_LAUNCHED(P);
  return KLDI_OK;
}

kldi_status launch_tau_combine(kldi_plan* P) {
  const int nb = (int)((P->n_pad + 255) / 256);
  k_tau_combine<<<nb, 256, 0, P->stream>>>(P->n_pad, P->d_drho_s, P->d_rho_s);
  KLDI_LAUNCHED(P);
  return KLDI_OK;
}

kldi_status launch_unpermute_rho(kldi_plan* P, double* rho, double* drho) {
  const int nb = (int)((P->n_pad + 255) / 256);
  k_unpermute_rho<<<nb, 256, 0, P->stream>>>(P->d_perm_g, P->n_pad, P->n_pts, P->d_rho_s, P->d_drho_s, rho, drho);
  KLDI_LAUNCHED(P);
  return KLDI_OK;
}

kldi_status launch_xc(kldi_plan* P, kldi_functional f) {
  const int nb = (int)((P->n_pad + 255) / 256);
  if (f == KLDI_GGA_PBEX)
    k_xc<true><<<nb, 256, 0, P->stream>>>(P->n_pad, P->d_rho_s, P->d_drho_s, P->d_gw, P->d_wv_s, P->d_epart);
  else
    k_xc<false><<<nb, 256, 0, P->stream>>>(P->n_pad, P->d_rho_s, nullptr, P->d_gw, P->d_wv_s, P->d_epart);
  KLDI_LAUNCHED(P);
  k_sum_partials<<<1, 1024, 0, P->stream>>>(P->d_epart, nb, P->d_E);
  KLDI_LAUNCHED(P);
  return KLDI_OK;
}

kldi_status launch_gather_wv(kldi_plan* P, const double* wv, bool gga, double scale) {
  const int nb = (int)((P->n_pad + 255) / 256);
  k_gather_wv<<<nb, 256, 0, P->stream>>>(P->d_perm_g, P->n_pad, P->n_pts, gga ? 4 : 1, wv, P->d_wv_s, scale);
  KLDI_LAUNCHED(P);
  return KLDI_OK;
}

kldi_status launch_finalise_V(kldi_plan* P, bool gga, double* V, int fixed) {
  dim3 grid((P->n_ao + 255) / 256, P->n_ao);
  const bool fx = (fixed < 0 ? P->v_mode == 2 : fixed != 0) && P->n_tasks > 0;
  if (gga && fx)
    k_finalise_V<true, true><<<grid, 256, 0, P->stream>>>(P->d_Vp, P->d_ao_perm, P->n_ao, V, P->d_fx);
  else if (gga)
    k_finalise_V<true, false><<<grid, 256, 0, P->stream>>>(P->d_Vp, P->d_ao_perm, P->n_ao, V, nullptr);
  else if (fx)
    k_finalise_V<false, true><<<grid, 256, 0, P->stream>>>(P->d_Vp, P->d_ao_perm, P->n_ao, V, P->d_fx);
  else
    k_finalise_V<false, false><<<grid, 256, 0, P->stream>>>(P->d_Vp, P->d_ao_perm, P->n_ao, V, nullptr);
  KLDI_LAUNCHED(P);
  return KLDI_OK;
}

}  // namespace kldi
