// C ABI entry points of libkldi (declared in include/kldi.h).
#include <algorithm>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <map>
#include <mutex>
#include <new>

#include "kldi_internal.h"
#include "ptx.cuh"

namespace kldi {
static thread_local char g_err[512] = "";
void set_error(const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
}

kldi_status ensure_smem_attr(const void* func, int bytes, int device) {
  static std::mutex mu;
  static std::map<const void*, uint64_t> done;  // kernel -> bitmask of devices that have the attribute
  std::lock_guard<std::mutex> lock(mu);
  uint64_t& m = done[func];
  if (device >= 0 && device < 64 && ((m >> device) & 1)) return KLDI_OK;
  KLDI_CUDA(cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
  if (device >= 0 && device < 64) m |= 1ull << device;
  return KLDI_OK;
}

// ------------------------------------------------------------------ FP64 pipe microbenchmark
__global__ void __launch_bounds__(256) k_peak_dmma(int iters, double* sink) {
  double c[16][2];
#pragma unroll
  for (int i = 0; i < 16; ++i) c[i][0] = c[i][1] = 0.0;
  double a = 1.0 + threadIdx.x * 1e-9, b = 1.0 - threadIdx.x * 1e-9;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 16; ++i) dmma884(c[i][0], c[i][1], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += c[i][0] + c[i][1];
  if (s == 123.456) sink[0] = s;
}
__global__ void __launch_bounds__(256) k_peak_dfma(int iters, double* sink) {
  double c[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) c[i] = i;
  double a = 1.0 + threadIdx.x * 1e-9, b = 1e-9 * threadIdx.x;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 16; ++i) c[i] = fma(c[i], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += c[i];
  if (s == 123.456) sink[0] = s;
}
// 16 DMMA + 64 DFMA per iteration: tells whether the tensor and the vector FP64 instructions share one pipe
__global__ void __launch_bounds__(256) k_peak_mix(int iters, double* sink) {
  double c[16][2], f[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) { c[i][0] = c[i][1] = 0.0; f[i] = i; }
  double a = 1.0 + threadIdx.x * 1e-9, b = 1.0 - threadIdx.x * 1e-9;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 16; ++i) {
      dmma884(c[i][0], c[i][1], a, b);
#pragma unroll
      for (int r = 0; r < 4; ++r) f[(4 * i + r) & 15] = fma(f[(4 * i + r) & 15], a, b);
    }
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += c[i][0] + c[i][1] + f[i];
  if (s == 123.456) sink[0] = s;
}
}  // namespace kldi

namespace kldi {
int g_default_ao_order = 0;
}

using namespace kldi;

extern "C" {

kldi_status kldi_set_plan_default(kldi_plan_default what, int value) {
  if (what != KLDI_DEFAULT_AO_ORDER || value < 0 || value > 2) {
    set_error("kldi_set_plan_default: unknown default %d or value %d", (int)what, value);
    return KLDI_EINVAL;
  }
  g_default_ao_order = value;
  return KLDI_OK;
}

kldi_status kldi_ao_order(const kldi_atoms* atoms, const kldi_shells* shells, int mode, int32_t* order, double* dist) {
  if (!atoms || !shells || !order || atoms->n_atoms <= 0 || mode != 1) {
    set_error("kldi_ao_order: null argument or unsupported mode");
    return KLDI_EINVAL;
  }
  for (int s = 0; s < shells->n_shells; ++s)
    if (shells->l[s] < 0 || shells->l[s] > 2 || shells->atom[s] < 0 || shells->atom[s] >= atoms->n_atoms) {
      set_error("kldi_ao_order: shell %d not supported", s);
      return KLDI_EINVAL;
    }
  std::vector<int> o;
  std::vector<double> d;
  if (!overlap_signature_order(atoms, shells, o, dist ? &d : nullptr)) {
    set_error("kldi_ao_order: more than 4096 centres");
    return KLDI_EINVAL;
  }
  for (int a = 0; a < atoms->n_atoms; ++a) order[a] = o[a];
  if (dist) std::copy(d.begin(), d.end(), dist);
  return KLDI_OK;
}

const char* kldi_last_error(void) { return g_err; }

uint64_t kldi_morton_key(const double* xyz, const double* origin) {
  if (!xyz || !origin) return ~0ull;
  return morton_key_host(xyz[0], xyz[1], xyz[2], origin[0], origin[1], origin[2]);
}

uint64_t kldi_grid_key(const double* xyz, const double* origin) {
  if (!xyz || !origin) return ~0ull;
  return grid_key_host(xyz[0], xyz[1], xyz[2], origin[0], origin[1], origin[2]);
}

kldi_status kldi_grid_keys(const double* xyz, int64_t n, const double* origin, uint64_t* keys) {
  if (!xyz || !origin || !keys || n < 0) {
    set_error("kldi_grid_keys: null argument");
    return KLDI_EINVAL;
  }
  for (int64_t i = 0; i < n; ++i)
    keys[i] = grid_key_host(xyz[3 * i], xyz[3 * i + 1], xyz[3 * i + 2], origin[0], origin[1], origin[2]);
  return KLDI_OK;
}

kldi_status kldi_plan_create(const kldi_atoms* atoms, const kldi_shells* shells, const kldi_grid* grid, double eps,
                             int want_gradients, void* cuda_stream, kldi_plan** out) {
  if (out) *out = nullptr;
  if (!atoms || !shells || !grid || !out || !atoms->xyz || !shells->atom || !shells->l || !shells->nprim_off ||
      !shells->alpha || !shells->coef || !grid->xyz || !grid->w || atoms->n_atoms <= 0 || shells->n_shells <= 0 ||
      grid->n_pts <= 0 || !(eps == eps)) {
    set_error("kldi_plan_create: null or empty argument");
    return KLDI_EINVAL;
  }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    set_error("kldi_plan_create: no CUDA device (this library has no CPU path)");
    return KLDI_ECUDA;
  }
  kldi_plan* P = new (std::nothrow) kldi_plan();
  if (!P) return KLDI_ENOMEM;
  P->stream = (cudaStream_t)cuda_stream;
  P->eps = eps;
  P->want_grad = want_gradients ? 1 : 0;
  cudaGetDevice(&P->device);
  cudaDeviceProp prop{};
  if (cudaGetDeviceProperties(&prop, P->device) != cudaSuccess || prop.major < 10) {
    set_error("kldi_plan_create: device is not sm_100+ (found sm_%d%d)", prop.major, prop.minor);
    delete P;
    return KLDI_ECUDA;
  }
  P->n_sm = prop.multiProcessorCount;
  kldi_status rc = plan_build(P, atoms, shells, grid);
  if (rc != KLDI_OK) {
    plan_free(P);
    delete P;
    return rc;
  }
  if (P->stats.max_k >= 32760) {
    set_error("kldi_plan_create: a grid block retains %lld AO columns (limit 32759)", (long long)P->stats.max_k);
    plan_free(P);
    delete P;
    return KLDI_EINVAL;
  }
  // FLOPs the rho kernel issues: full form, and the triangular-D form (mirrors the producer loop of k_rho)
  double fr = 0, frs = 0;
  for (int64_t p = 0; p < P->n_blocks; ++p) {
    const int k8 = (int)(P->h_panel_off[p + 1] - P->h_panel_off[p]);
    fr += 2.0 * GB * (double)k8 * k8;
    if (!k8) continue;
    const int ntile = (k8 + 127) / 128, W = (((k8 + ntile - 1) / ntile) + 31) & ~31;
    for (int jt = 0; jt < ntile; ++jt) {
      const int n0 = jt * W, Wj = std::min(W, k8 - n0);
      for (int k0 = n0; k0 < k8; k0 += 32) {
        const int kc = std::min(32, k8 - k0);
        if (k0 < n0 + Wj) {  // diagonal chunk: rectangle before the own columns + the own block, 8-row k-step pairs m reach own groups <= m
          const int nown = kc >> 3;
          frs += 2.0 * GB * ((double)kc * (k0 - n0) + 32.0 * nown * (nown + 1));
        } else {
          frs += 2.0 * GB * kc * (double)Wj;
        }
      }
    }
  }
  P->stats.flops_rho_exec = fr;
  P->stats.flops_rho_exec_sym = frs;
  *out = P;
  return KLDI_OK;
}

kldi_status kldi_plan_destroy(kldi_plan* P) {
  if (!P) return KLDI_OK;
  DeviceGuard dev_guard(P->device);
  plan_free(P);
  delete P;
  return KLDI_OK;
}

kldi_status kldi_plan_stats(const kldi_plan* P, kldi_stats* out) {
  if (!P || !out) {
    set_error("kldi_plan_stats: null argument");
    return KLDI_EINVAL;
  }
  DeviceGuard dev_guard(P->device);
  *out = P->stats;
  out->kernel_launches = P->launches;
  out->pair_stages_total = out->pair_stages_executed = -1;
  if (P->pair_counts_valid) {  // counters of the most recent rho contraction run with KLDI_OPT_PAIR_TEST
    unsigned long long c[2] = {0, 0};
    KLDI_CUDA(cudaStreamSynchronize(P->stream));
    KLDI_CUDA(cudaMemcpy(c, P->d_pcount, sizeof(c), cudaMemcpyDeviceToHost));
    out->pair_stages_total = (int64_t)c[0];
    out->pair_stages_executed = (int64_t)c[1];
  }
  return KLDI_OK;
}

#define EV(i) KLDI_CUDA(cudaEventRecord(P->ev[i], P->stream))

kldi_status kldi_eval_rho(kldi_plan* P, const double* D, double* rho, double* drho) {
  if (!P || !D || !rho) {
    set_error("kldi_eval_rho: null argument");
    return KLDI_EINVAL;
  }
  DeviceGuard dev_guard(P->device);
  if (drho && !P->want_grad) {
    set_error("kldi_eval_rho: gradients requested from a plan created with want_gradients = 0");
    return KLDI_ESTATE;
  }
  kldi_status rc;
  P->have_timings = false;
  P->launches = 0;
  EV(0);
  if ((rc = launch_permute_D(P, D, drho != nullptr)) != KLDI_OK) return rc;
  EV(1);
  if ((rc = launch_rho(P, drho != nullptr)) != KLDI_OK) return rc;
  EV(2);
  if ((rc = launch_unpermute_rho(P, rho, drho)) != KLDI_OK) return rc;
  for (int i = 3; i < 7; ++i) EV(i);
  P->have_timings = true;
  return KLDI_OK;
}

kldi_status kldi_build_vxc(kldi_plan* P, const double* wv, int gga, double* V) {
  if (!P || !wv || !V) {
    set_error("kldi_build_vxc: null argument");
    return KLDI_EINVAL;
  }
  DeviceGuard dev_guard(P->device);
  if (gga && !P->want_grad) {
    set_error("kldi_build_vxc: GGA form requested from a plan created with want_gradients = 0");
    return KLDI_ESTATE;
  }
  kldi_status rc;
  P->have_timings = false;
  P->launches = 0;
  for (int i = 0; i < 4; ++i) EV(i);
  if ((rc = launch_gather_wv(P, wv, gga != 0)) != KLDI_OK) return rc;
  EV(4);
  if ((rc = launch_vxc(P, gga != 0)) != KLDI_OK) return rc;
  EV(5);
  if ((rc = launch_finalise_V(P, gga != 0, V)) != KLDI_OK) return rc;
  EV(6);
  P->have_timings = true;
  return KLDI_OK;
}

static kldi_status exc_enqueue(kldi_plan* P, const double* D, kldi_functional f, double* V) {
  const bool gga = (f == KLDI_GGA_PBEX);
  kldi_status rc;
  P->have_timings = false;
  P->launches = 0;
  EV(0);
  if ((rc = launch_permute_D(P, D, gga)) != KLDI_OK) return rc;
  EV(1);
  if ((rc = launch_rho(P, gga)) != KLDI_OK) return rc;
  EV(2);
  if ((rc = launch_xc(P, f)) != KLDI_OK) return rc;
  EV(3);
  EV(4);
  if (V) {
    if ((rc = launch_vxc(P, gga)) != KLDI_OK) return rc;
    EV(5);
    if ((rc = launch_finalise_V(P, gga, V)) != KLDI_OK) return rc;
  } else {
    EV(5);
  }
  EV(6);
  KLDI_CUDA(cudaMemcpyAsync(P->h_E, P->d_E, sizeof(double), cudaMemcpyDeviceToHost, P->stream));
  P->have_timings = true;
  return KLDI_OK;
}

kldi_status kldi_exc(kldi_plan* P, const double* D, kldi_functional f, double* Exc, double* V) {
  if (!P || !D || !Exc || (f != KLDI_LDA_SLATER && f != KLDI_GGA_PBEX)) {
    set_error("kldi_exc: null argument or unknown functional");
    return KLDI_EINVAL;
  }
  DeviceGuard dev_guard(P->device);
  if (f == KLDI_GGA_PBEX && !P->want_grad) {
    set_error("kldi_exc: GGA functional needs a plan created with want_gradients = 1");
    return KLDI_ESTATE;
  }
  kldi_status rc = exc_enqueue(P, D, f, V);
  if (rc != KLDI_OK) return rc;
  KLDI_CUDA(cudaStreamSynchronize(P->stream));
  *Exc = *P->h_E;
  return KLDI_OK;
}

kldi_status kldi_exc_host(kldi_plan* P, const double* D_host, kldi_functional f, double* Exc, double* V_host) {
  if (!P || !D_host || !Exc || (f != KLDI_LDA_SLATER && f != KLDI_GGA_PBEX)) {
    set_error("kldi_exc_host: null argument or unknown functional");
    return KLDI_EINVAL;
  }
  DeviceGuard dev_guard(P->device);
  if (f == KLDI_GGA_PBEX && !P->want_grad) {
    set_error("kldi_exc_host: GGA functional needs a plan created with want_gradients = 1");
    return KLDI_ESTATE;
  }
  const size_t nn = sizeof(double) * (size_t)P->n_ao * P->n_ao;
  if (!P->d_stage_host) KLDI_CUDA(cudaMalloc(&P->d_stage_host, 2 * nn));
  double* dD = P->d_stage_host;
  double* dV = V_host ? P->d_stage_host + (size_t)P->n_ao * P->n_ao : nullptr;
  // D is symmetric and k_permute_D reads only its lower triangle: upload that half, in 32 row bands (band [r0, r1)
  // needs the columns [0, r1)), 52 % of the bytes of the full matrix over PCIe
  {
    const int n = P->n_ao, nb = n < 1024 ? 1 : 32;
    for (int b = 0; b < nb; ++b) {
      const int r0 = (int)((int64_t)n * b / nb), r1 = (int)((int64_t)n * (b + 1) / nb);
      if (r1 > r0)
        KLDI_CUDA(cudaMemcpy2DAsync(dD + (size_t)r0 * n, sizeof(double) * n, D_host + (size_t)r0 * n,
                                    sizeof(double) * n, sizeof(double) * r1, r1 - r0, cudaMemcpyHostToDevice,
                                    P->stream));
    }
  }
  kldi_status rc = exc_enqueue(P, dD, f, dV);
  if (rc != KLDI_OK) return rc;
  if (V_host && P->host_v_triangle) {
    // V is exactly symmetric: download the lower triangle only, in the same 32 row bands as the upload of D
    const int n = P->n_ao, nb = n < 1024 ? 1 : 32;
    for (int b = 0; b < nb; ++b) {
      const int r0 = (int)((int64_t)n * b / nb), r1 = (int)((int64_t)n * (b + 1) / nb);
      if (r1 > r0)
        KLDI_CUDA(cudaMemcpy2DAsync(V_host + (size_t)r0 * n, sizeof(double) * n, dV + (size_t)r0 * n, sizeof(double) * n,
                                    sizeof(double) * r1, r1 - r0, cudaMemcpyDeviceToHost, P->stream));
    }
  } else if (V_host) {
    KLDI_CUDA(cudaMemcpyAsync(V_host, dV, nn, cudaMemcpyDeviceToHost, P->stream));
  }
  KLDI_CUDA(cudaStreamSynchronize(P->stream));
  *Exc = *P->h_E;
  return KLDI_OK;
}

kldi_status kldi_eval_tau(kldi_plan* P, const double* D, double* tau) {
  if (!P || !D || !tau) {
    set_error("kldi_eval_tau: null argument");
    return KLDI_EINVAL;
  }
  DeviceGuard dev_guard(P->device);
  if (!P->want_grad) {
    set_error("kldi_eval_tau: needs a plan created with want_gradients = 1 (the stores of grad Phi)");
    return KLDI_ESTATE;
  }
  kldi_status rc;
  P->have_timings = false;
  P->launches = 0;
  EV(0);
  if ((rc = launch_permute_D(P, D, false)) != KLDI_OK) return rc;  // triangular D': the product is symmetric in mu, nu
  EV(1);
  if (P->rho_impl == 2) {  // KLDI_OPT_RHO_TC: the three builds as int8 slice products on tcgen05
    if ((rc = launch_tau_tc(P)) != KLDI_OK) return rc;
  } else {
    for (int c = 0; c < 3; ++c)
      if ((rc = launch_rho_lda_on(P, P->d_dphi[c], P->d_drho_s + (size_t)c * P->n_pad)) != KLDI_OK) return rc;
  }
  if ((rc = launch_tau_combine(P)) != KLDI_OK) return rc;
  EV(2);
  if ((rc = launch_unpermute_rho(P, tau, nullptr)) != KLDI_OK) return rc;
  for (int i = 3; i < 7; ++i) EV(i);
  P->have_timings = true;
  return KLDI_OK;
}

kldi_status kldi_build_vtau(kldi_plan* P, const double* wv_tau, double* V) {
  if (!P || !wv_tau || !V) {
    set_error("kldi_build_vtau: null argument");
    return KLDI_EINVAL;
  }
  DeviceGuard dev_guard(P->device);
  if (!P->want_grad) {
    set_error("kldi_build_vtau: needs a plan created with want_gradients = 1 (the stores of grad Phi)");
    return KLDI_ESTATE;
  }
  kldi_status rc;
  P->have_timings = false;
  P->launches = 0;
  for (int i = 0; i < 4; ++i) EV(i);
  if ((rc = launch_gather_wv(P, wv_tau, false, 0.5)) != KLDI_OK) return rc;
  EV(4);
  if ((rc = launch_vtau(P)) != KLDI_OK) return rc;
  EV(5);
  if ((rc = launch_finalise_V(P, false, V, P->v_mode != 0)) != KLDI_OK) return rc;
  EV(6);
  P->have_timings = true;
  return KLDI_OK;
}

kldi_status kldi_exc_grad(kldi_plan* P, const double* D, kldi_functional f, double* Exc, double* grad) {
  if (!P || !D || !grad) {
    set_error("kldi_exc_grad: null argument");
    return KLDI_EINVAL;
  }
  DeviceGuard dev_guard(P->device);
  if (f != KLDI_LDA_SLATER && f != KLDI_GGA_PBEX) {
    set_error("kldi_exc_grad: unknown functional");
    return KLDI_EINVAL;
  }
  if (!P->want_grad) {
    set_error("kldi_exc_grad: needs a plan created with want_gradients = 1 (the stores of grad Phi)");
    return KLDI_ESTATE;
  }
  const bool gga = f == KLDI_GGA_PBEX;
  const size_t store = sizeof(double) * GB * (size_t)(P->total_cols + 64);
  if (!P->d_x) KLDI_CUDA(cudaMalloc(&P->d_x, store));
  if (gga && !P->d_xd) KLDI_CUDA(cudaMalloc(&P->d_xd, 3 * store + sizeof(double) * P->n_pad));
  kldi_status rc;
  P->have_timings = false;
  P->launches = 0;
  EV(0);
  if ((rc = launch_permute_D(P, D, true)) != KLDI_OK) return rc;  // full D: the gradient needs X = Phi D itself
  EV(1);
  // LDA: X-only form (rho + X).  GGA: the GGA form (rho, grad rho and X in one pass), then X^d = d_d Phi D
  // KLDI_OPT_RHO_TC: the X-only builds (LDA: X = Phi D; GGA: the three X^d) run as int8 slice products on tcgen05
  const bool tc = P->rho_impl == 2 && !P->pair_test;
  if (!gga && tc) {
    if ((rc = launch_x_tc(P, 0, P->d_x, P->d_rho_s, true)) != KLDI_OK) return rc;
  } else if ((rc = launch_rho(P, true, P->d_x, !gga)) != KLDI_OK) {
    return rc;
  }
  if (gga) {
    double* scratch = P->d_xd + 3 * (store / sizeof(double));
    for (int d = 0; d < 3; ++d) {
      double* xd = P->d_xd + d * (store / sizeof(double));
      rc = tc ? launch_x_tc(P, 1 + d, xd, scratch, d == 0) : launch_x_on(P, P->d_dphi[d], xd, scratch);
      if (rc != KLDI_OK) return rc;
    }
  }
  EV(2);
  if ((rc = launch_xc(P, f)) != KLDI_OK) return rc;
  EV(3);
  EV(4);
  if ((rc = gga ? launch_grad_cols_gga(P, grad) : launch_grad_cols(P, grad)) != KLDI_OK) return rc;
  EV(5);
  EV(6);
  KLDI_CUDA(cudaMemcpyAsync(P->h_E, P->d_E, sizeof(double), cudaMemcpyDeviceToHost, P->stream));
  P->have_timings = true;
  KLDI_CUDA(cudaStreamSynchronize(P->stream));
  if (Exc) *Exc = *P->h_E;
  return KLDI_OK;
}

kldi_status kldi_plan_set_option(kldi_plan* P, kldi_option option, int value) {
  if (!P || (option != KLDI_OPT_DETERMINISTIC_V && option != KLDI_OPT_PAIR_TEST && option != KLDI_OPT_RHO_DFMA &&
             option != KLDI_OPT_RHO_TC && option != KLDI_OPT_HOST_V_TRIANGLE)) {
    set_error("kldi_plan_set_option: null plan or unknown option %d", (int)option);
    return KLDI_EINVAL;
  }
  if (option == KLDI_OPT_DETERMINISTIC_V) {
    if (value < 0 || value > 2) {
      set_error("kldi_plan_set_option: KLDI_OPT_DETERMINISTIC_V takes 0, 1 or 2");
      return KLDI_EINVAL;
    }
    P->v_mode = value;
  }
  if (option == KLDI_OPT_RHO_DFMA) P->rho_impl = value ? 1 : 0;
  if (option == KLDI_OPT_RHO_TC) P->rho_impl = value ? 2 : 0;
  if (option == KLDI_OPT_HOST_V_TRIANGLE) P->host_v_triangle = value ? 1 : 0;
  if (option == KLDI_OPT_PAIR_TEST) {
    P->pair_test = value ? 1 : 0;
    if (!value) P->pair_counts_valid = false;
  }
  return KLDI_OK;
}

kldi_status kldi_last_timings(kldi_plan* P, double* out) {
  if (!P || !out) {
    set_error("kldi_last_timings: null argument");
    return KLDI_EINVAL;
  }
  DeviceGuard dev_guard(P->device);
  if (!P->have_timings) {
    set_error("kldi_last_timings: no completed call on this plan");
    return KLDI_ESTATE;
  }
  KLDI_CUDA(cudaStreamSynchronize(P->stream));
  for (int i = 0; i < 6; ++i) {
    float ms = 0.f;
    KLDI_CUDA(cudaEventElapsedTime(&ms, P->ev[i], P->ev[i + 1]));
    out[i] = ms;
  }
  float ms = 0.f;
  KLDI_CUDA(cudaEventElapsedTime(&ms, P->ev[0], P->ev[6]));
  out[6] = ms;
  out[7] = 0.0;
  return KLDI_OK;
}

kldi_status kldi_plan_export(const kldi_plan* P, int which, void* buf, int64_t cap, int64_t* need) {
  if (!P || !need) {
    set_error("kldi_plan_export: null argument");
    return KLDI_EINVAL;
  }
  DeviceGuard dev_guard(P->device);
  const void* hsrc = nullptr;
  const void* dsrc = nullptr;
  int64_t bytes = 0;
  switch (which) {
    case 0: dsrc = P->d_perm_g; bytes = 4 * P->n_pad; break;
    case 1: hsrc = P->h_row_ptr.data(); bytes = 4 * (int64_t)P->h_row_ptr.size(); break;
    case 2: hsrc = P->h_col_idx.data(); bytes = 4 * (int64_t)P->h_col_idx.size(); break;
    case 3: hsrc = P->h_col_ptr.data(); bytes = 4 * (int64_t)P->h_col_ptr.size(); break;
    case 4: hsrc = P->h_row_idx.data(); bytes = 4 * (int64_t)P->h_row_idx.size(); break;
    case 5: hsrc = P->h_pos.data(); bytes = 4 * (int64_t)P->h_pos.size(); break;
    case 6: hsrc = P->h_shell_perm.data(); bytes = 4 * (int64_t)P->h_shell_perm.size(); break;
    case 7: hsrc = P->h_ao_perm.data(); bytes = 4 * (int64_t)P->h_ao_perm.size(); break;
    case 8: dsrc = P->d_keys; bytes = 8 * P->n_pad; break;
    case 9: dsrc = P->d_blk_amax; bytes = 8 * (int64_t)P->h_col_idx.size(); break;
    case 10: hsrc = P->h_panel_off.data(); bytes = 8 * (int64_t)P->h_panel_off.size(); break;
    case 11: hsrc = P->h_blk_col0.data(); bytes = 4 * (int64_t)P->h_blk_col0.size(); break;
    default: set_error("kldi_plan_export: unknown array %d", which); return KLDI_EINVAL;
  }
  *need = bytes;
  if (!buf) return KLDI_OK;
  if (cap < bytes) {
    set_error("kldi_plan_export: buffer too small (%lld < %lld)", (long long)cap, (long long)bytes);
    return KLDI_EINVAL;
  }
  if (hsrc) {
    memcpy(buf, hsrc, (size_t)bytes);
  } else {
    KLDI_CUDA(cudaStreamSynchronize(P->stream));
    KLDI_CUDA(cudaMemcpy(buf, dsrc, (size_t)bytes, cudaMemcpyDeviceToHost));
  }
  return KLDI_OK;
}

kldi_status kldi_plan_export_tile(const kldi_plan* P, int64_t entry, int c, double* out, int64_t cap, int32_t* width) {
  if (!P || !out || !width || entry < 0 || entry >= (int64_t)P->h_col_idx.size() || c < 0 || c > 3 ||
      (c > 0 && !P->want_grad)) {
    set_error("kldi_plan_export_tile: bad argument");
    return KLDI_EINVAL;
  }
  DeviceGuard dev_guard(P->device);
  // grid block of the entry: binary search in row_ptr
  int64_t lo = 0, hi = P->n_blocks;
  while (hi - lo > 1) {
    const int64_t mid = (lo + hi) / 2;
    if (P->h_row_ptr[mid] <= entry) lo = mid; else hi = mid;
  }
  const int64_t p = lo;
  const int32_t c0 = P->h_blk_col0[entry];
  const int32_t c1 = (entry + 1 < P->h_row_ptr[p + 1]) ? P->h_blk_col0[entry + 1] : -1;
  int32_t w;
  if (c1 >= 0) {
    w = c1 - c0;
  } else {  // last block of the row: width from the shell table is not on the host; use K_p
    int32_t kp = 0;
    KLDI_CUDA(cudaMemcpy(&kp, P->d_kp + p, sizeof(int32_t), cudaMemcpyDeviceToHost));
    w = kp - c0;
  }
  *width = w;
  const int64_t bytes = (int64_t)w * GB * 8;
  if (cap < bytes) {
    set_error("kldi_plan_export_tile: buffer too small");
    return KLDI_EINVAL;
  }
  const double* src = (c == 0 ? P->d_phi : P->d_dphi[c - 1]) + (P->h_panel_off[p] + c0) * GB;
  KLDI_CUDA(cudaStreamSynchronize(P->stream));
  KLDI_CUDA(cudaMemcpy(out, src, (size_t)bytes, cudaMemcpyDeviceToHost));
  return KLDI_OK;
}

kldi_status kldi_fp64_peak(int kind, int iters, double* tflops) {
  if (!tflops || iters <= 0) {
    set_error("kldi_fp64_peak: bad argument");
    return KLDI_EINVAL;
  }
  int dev = 0, nsm = 0;
  KLDI_CUDA(cudaGetDevice(&dev));
  KLDI_CUDA(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
  double* sink = nullptr;
  KLDI_CUDA(cudaMalloc(&sink, 8));
  cudaEvent_t e0, e1;
  KLDI_CUDA(cudaEventCreate(&e0));
  KLDI_CUDA(cudaEventCreate(&e1));
  const int grid = nsm * 4;
  for (int rep = 0; rep < 2; ++rep) {  // first pass warms up
    KLDI_CUDA(cudaEventRecord(e0));
    if (kind == 0)
      k_peak_dmma<<<grid, 256>>>(iters, sink);
    else if (kind == 1)
      k_peak_dfma<<<grid, 256>>>(iters, sink);
    else
      k_peak_mix<<<grid, 256>>>(iters, sink);
    KLDI_CUDA(cudaEventRecord(e1));
    KLDI_CUDA(cudaEventSynchronize(e1));
  }
  float ms = 0.f;
  KLDI_CUDA(cudaEventElapsedTime(&ms, e0, e1));
  const double per_thread_block = (kind == 0)   ? 8.0 * 16 * 2 * 8 * 8 * 4
                                  : (kind == 1) ? 256.0 * 16 * 2
                                                : 8.0 * 16 * 2 * 8 * 8 * 4 + 256.0 * 64 * 2;  // flops per CTA per iter
  *tflops = per_thread_block * iters * grid / (ms * 1e-3) / 1e12;
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(sink);
  return KLDI_OK;
}

}  // extern "C"
