// Internal declarations of libkldi (not part of the ABI).  sm_100a only.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "kldi.h"

namespace kldi {

constexpr int GB = 128;  // points per grid block (BASELINE.json; PAPER.md:118 uses d = 32)

void set_error(const char* fmt, ...);

// "V layout" of a panel (second copy of Phi, and Z, read by the V contraction): 4 slabs of 32 grid rows; slab
// rc holds [K8 columns][32 rows] contiguously, so any column interval of a slab is ONE bulk copy; inside a
// column the 16-byte chunk c (rows 2c, 2c+1) sits at chunk c ^ (col & 7), which makes the 16-byte MMA
// fragment loads of 8 adjacent columns bank-conflict free without padding (the smem image is the HBM image).
constexpr int V_SLAB = 32;  // grid rows per slab of the V layout = MMA K rows per ring stage of k_vgram
__host__ __device__ __forceinline__ int64_t vlayout_off(int64_t panel_off_p, int K8, int col, int row) {
  const int rc = row / V_SLAB, rr = row % V_SLAB, c = rr >> 1;
  return panel_off_p * GB + (int64_t)rc * K8 * V_SLAB + (int64_t)col * V_SLAB + (((c ^ (col & 7)) << 1) | (rr & 1));
}

// Fixed-point scale of the V accumulation: the power of two that maps |x| <= bound below 2^61.
__host__ __device__ __forceinline__ double fx_scale(double bound) {
  if (!(bound > 0.0)) return 1.0;
  const int e = 60 - ilogb(bound);
  return scalbn(1.0, e > 1000 ? 1000 : e);  // a denormal-small bound would overflow the scale
}

#define KLDI_CUDA(call)                                                                     \
  do {                                                                                      \
    cudaError_t e__ = (call);                                                               \
    if (e__ != cudaSuccess) {                                                               \
      kldi::set_error("%s:%d: %s -> %s", __FILE__, __LINE__, #call, cudaGetErrorString(e__)); \
      return e__ == cudaErrorMemoryAllocation ? KLDI_ENOMEM : KLDI_ECUDA;                   \
    }                                                                                       \
  } while (0)

// The > 48 KB dynamic-shared-memory opt-in belongs to the device's context: remember per (kernel, device), thread-safe.
kldi_status ensure_smem_attr(const void* func, int bytes, int device);

// A plan is bound to the device that was current at kldi_plan_create; every entry point runs with that device
// current and restores the caller's on return.
struct DeviceGuard {
  int prev = -1;
  bool switched = false;
  explicit DeviceGuard(int device) {
    if (cudaGetDevice(&prev) == cudaSuccess && prev != device) switched = cudaSetDevice(device) == cudaSuccess;
  }
  ~DeviceGuard() {
    if (switched) cudaSetDevice(prev);
  }
};

// after a kernel launch on plan P: check the launch and count it (kldi_stats.kernel_launches)
#define KLDI_LAUNCHED(P)               \
  do {                                 \
    KLDI_CUDA(cudaGetLastError());     \
    ++(P)->launches;                   \
  } while (0)

// Device-side view of the basis in the plan's spatial shell order.
struct ShellTable {
  const double* atom_xyz;    // [n_atoms][3]
  const int32_t* sh_atom;    // [n_shells]
  const int32_t* sh_l;       // [n_shells]
  const int32_t* sh_prim0;   // [n_shells+1]
  const int32_t* sh_ao0;     // [n_shells+1] first plan-order AO of the shell
  const double* prim_alpha;  // [n_prim]
  const double* prim_cn;     // [n_prim] coef * (2a/pi)^{3/4} (4a)^{l/2}
};

}  // namespace kldi

struct kldi_plan {
  cudaStream_t stream = nullptr;
  int device = 0, n_sm = 0;
  double eps = 0.0;
  int want_grad = 0;
  int32_t n_atoms = 0, n_shells = 0, n_ao = 0, n_prim = 0;
  int64_t n_pts = 0, n_blocks = 0, n_pad = 0;
  kldi_stats stats{};

  // ---- basis (device), plan order
  double* d_atom_xyz = nullptr;
  int32_t *d_sh_atom = nullptr, *d_sh_l = nullptr, *d_sh_prim0 = nullptr, *d_sh_ao0 = nullptr;
  double *d_prim_alpha = nullptr, *d_prim_cn = nullptr;
  int32_t *d_shell_perm = nullptr, *d_ao_perm = nullptr;  // plan index -> caller index
  int32_t* d_ao_atom = nullptr;                           // plan AO -> plan atom rank
  int32_t* d_ao_atom_c = nullptr;                         // plan AO -> caller atom index (nuclear gradient)

  // ---- grid (device), Morton order, SoA, padded to n_pad = n_blocks*128
  double *d_gx = nullptr, *d_gy = nullptr, *d_gz = nullptr, *d_gw = nullptr;
  int32_t* d_perm_g = nullptr;  // sorted -> caller, -1 = padding
  uint64_t* d_keys = nullptr;

  // ---- BCS(R) / BCS(C)
  int32_t *d_row_ptr = nullptr, *d_col_idx = nullptr, *d_blk_col0 = nullptr;
  int32_t *d_col_ptr = nullptr, *d_row_idx = nullptr, *d_pos = nullptr;
  double* d_blk_amax = nullptr;
  int64_t* d_panel_off = nullptr;  // [n_blocks+1] packed-column offsets (each K_p padded to 8)
  int32_t *d_kp = nullptr;         // [n_blocks] K_p (unpadded)
  int32_t* d_colidx = nullptr;     // [total_cols] plan AO index of every packed column (pad -> 0)
  int64_t total_cols = 0;
  double* d_phi = nullptr;         // [total_cols + slack][128] column-major tiles
  double* d_dphi[3] = {nullptr, nullptr, nullptr};
  double* d_phi_v = nullptr;       // second copy of Phi in the V layout (vlayout_off)
  double* d_dphi_v[3] = {nullptr, nullptr, nullptr};  // gradient stores in the V layout (kldi_build_vtau, first use)
  double* d_z = nullptr;           // GGA: Z = 1/2 wv0 Phi + sum_c wv_c d_c Phi, V layout
  double* d_x = nullptr;           // nuclear gradient: X = Phi D of every panel, rho layout, allocated on first use
  double* d_xd = nullptr;          // GGA nuclear gradient: X^d = d_d Phi D, d = x, y, z (three stores) + [n_pad] scratch

  // ---- V contraction schedule (vsched.h), index 0: LDA upper triangle, 1: GGA square
  int32_t* d_vsched_ptr[2] = {nullptr, nullptr};  // [max_nb + 2] first pass of an nb-block panel
  void* d_vpasses[2] = {nullptr, nullptr};
  void* d_vitems[2] = {nullptr, nullptr};
  int64_t* d_gram_off[2] = {nullptr, nullptr};    // [n_blocks + 1] workspace offsets of G_p (deterministic mode)
  int64_t gram_elems[2] = {0, 0};
  double* d_gram = nullptr;                       // lazily allocated workspace of G_p partials
  int64_t gram_cap = 0;
  int32_t* d_ao_shell = nullptr;                  // plan AO -> plan shell
  int rho_impl = 0;                               // LDA rho build: 0 DMMA tiles, 1 DFMA register tiles (KLDI_OPT_RHO_DFMA),
                                                  // 2 int8 slice products on tcgen05 (KLDI_OPT_RHO_TC)
  // ---- int8 slice-product path (rho_i8.cu), allocated on first use
  unsigned char* d_phiq = nullptr;                // [tc_chunks][NSL][4096] digit planes of Phi, tensor-core smem image
  double* d_sigma = nullptr;                      // [n_pad] row scales of the digit planes
  unsigned char* d_dphiq[3] = {nullptr, nullptr, nullptr};  // the same for the gradient stores (kldi_eval_tau, first use)
  double* d_dsigma[3] = {nullptr, nullptr, nullptr};
  bool dq_upper_dirty = false;                    // the last digit split wrote the upper triangle of Dq (full-D form)
  unsigned long long* d_Dq = nullptr;             // [n_ao][n_ao] packed digits of D' (per call)
  double* d_tau = nullptr;                        // [2][n_ao] column scales of D', column maxima
  int64_t* d_chunk_off = nullptr;                 // [n_blocks+1] first 32-column chunk of grid block p
  int64_t tc_chunks = 0;
  int v_mode = 2;                                 // 0: red.global.add.f64 epilogue, 1: workspace + fixed-order reduce,
                                                  // 2: 64-bit fixed-point integer atomics (reproducible)
  double* d_fx = nullptr;                         // [1 + n_blocks] fixed-point bound, then s_p = sum_g |wv_g| per block
  // ---- executable-pair selection (pairsel.cu), allocated on first use
  int pair_test = 0;
  double* d_bmax = nullptr;                       // [n_shells][n_shells] b_qr = max|D_qr|
  unsigned long long* d_pmask = nullptr;          // [n_blocks] stage masks, then 2 counters
  unsigned long long* d_pcount = nullptr;         // -> d_pmask + n_blocks: {stages without the test, stages executed}
  bool pair_counts_valid = false;

  // ---- task lists
  int32_t* d_tasks = nullptr;  // non-empty grid blocks in Morton order
  int32_t n_tasks = 0;
  int32_t* d_ticket = nullptr;  // [4] atomic work counters

  // ---- per-call buffers
  double *d_Dp = nullptr, *d_Vp = nullptr;  // plan-order D and V accumulators [n_ao][n_ao]
  double *d_rho_s = nullptr, *d_drho_s = nullptr, *d_wv_s = nullptr;  // sorted order, [n_pad], [3][n_pad], [4][n_pad]
  double *d_epart = nullptr, *d_E = nullptr;
  double* d_stage_host = nullptr;  // device staging for kldi_exc_host: D and V
  double* h_E = nullptr;           // pinned
  cudaEvent_t ev[8] = {};
  bool have_timings = false;
  int64_t launches = 0;            // kernels launched by the current / most recent compute call
  int host_v_triangle = 0;         // KLDI_OPT_HOST_V_TRIANGLE

  // ---- host copies kept for export / tests
  std::vector<int32_t> h_row_ptr, h_col_idx, h_blk_col0, h_col_ptr, h_row_idx, h_pos, h_shell_perm, h_ao_perm;
  std::vector<int64_t> h_panel_off;
};

namespace kldi {
// plan.cu
uint64_t morton_key_host(double x, double y, double z, double x0, double y0, double z0);
uint64_t grid_key_host(double x, double y, double z, double x0, double y0, double z0);
kldi_status plan_build(kldi_plan* P, const kldi_atoms* atoms, const kldi_shells* shells, const kldi_grid* grid);
void plan_free(kldi_plan* P);
// aoorder.cu: atom order by overlap-signature clustering; dist_out: the cosine distances
bool overlap_signature_order(const kldi_atoms* atoms, const kldi_shells* shells, std::vector<int>& order,
                             std::vector<double>* dist_out = nullptr);
extern int g_default_ao_order;  // kldi_set_plan_default(KLDI_DEFAULT_AO_ORDER): 0 curve, 1 overlap signature, 2 caller
// contract.cu
kldi_status launch_permute_D(kldi_plan* P, const double* D, bool gga);
// pairsel.cu
kldi_status launch_pair_select(kldi_plan* P, bool tri);
kldi_status launch_rho(kldi_plan* P, bool gga, double* x_store = nullptr, bool x_only = true);
kldi_status launch_x_on(kldi_plan* P, const double* store, double* x_out, double* rho_scratch);
kldi_status launch_grad_cols_gga(kldi_plan* P, double* grad);
// rho_i8.cu
kldi_status launch_rho_tc(kldi_plan* P);
kldi_status launch_tau_tc(kldi_plan* P);
kldi_status launch_x_tc(kldi_plan* P, int which, double* x_out, double* rho_out, bool slice_d);  // t_c = rowsum(d_c Phi o d_c Phi D') for c = x, y, z into d_drho_s (D' in d_Dp)
kldi_status launch_grad_cols(kldi_plan* P, double* grad);
kldi_status launch_unpermute_rho(kldi_plan* P, double* rho, double* drho);
kldi_status launch_xc(kldi_plan* P, kldi_functional f);
kldi_status launch_gather_wv(kldi_plan* P, const double* wv, bool gga, double scale = 1.0);
kldi_status launch_rho_lda_on(kldi_plan* P, const double* store, double* out_s);
kldi_status launch_tau_combine(kldi_plan* P);
kldi_status launch_vtau(kldi_plan* P);
kldi_status launch_vxc(kldi_plan* P, bool gga);
kldi_status launch_finalise_V(kldi_plan* P, bool gga, double* V, int fixed = -1);  // fixed: -1 = by v_mode
// vgram.cu
kldi_status vsched_upload(kldi_plan* P, const std::vector<int32_t>& h_kp, const std::vector<int32_t>& h_sh_ao0);
}  // namespace kldi
