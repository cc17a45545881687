// kldi_xc_lda_noalloc: the functional + energy step (H3: Slater exchange per point, wv = w v_rho, E_xc = sum_g w_g e_g,
// PAPER.md:57-63 Eq. 1, 71 Eq. 3) as an entry point that ALLOCATES NOTHING — for callers that cannot call cudaMalloc
// (CUDA graph capture, tight serving loops, harnesses that forbid it).  It is a variant of k_xc (contract.cu), whose
// per-block energy partials live in a plan-owned buffer; here they live in a file-scope static __device__ array of a
// fixed maximum size, so the call needs no plan and no allocation.  The existing code paths are untouched.
//
// The array is shared by every call on a device and keeps the last call's contents: a call overwrites the partials it
// then sums (nothing has to start at zero), and calls that overlap on the GPU (different streams) race on it.
#include <mutex>

#include "kldi_internal.h"

namespace kldi {
namespace {

constexpr int64_t NOALLOC_MAX_PTS = 8388608;                 // 2^23 grid points per call
constexpr int NOALLOC_TPB = 256;
constexpr int NOALLOC_MAX_PART = (int)(NOALLOC_MAX_PTS / NOALLOC_TPB);  // 32,768 partials = 256 KB per GPU
static __device__ __align__(256) double g_xc_partials[NOALLOC_MAX_PART];

constexpr double C_X = 0.73855876638202240588;  // (3/4)(3/pi)^{1/3}
constexpr double RHO_CUT = 1e-20;               // reading A9: below this density e = v = 0

// one thread per point; fixed reduction tree per block -> part[blockIdx.x] (bitwise reproducible)
__global__ void __launch_bounds__(NOALLOC_TPB) k_xc_lda_static(int64_t n, const double* __restrict__ rho,
                                                               const double* __restrict__ w, double* __restrict__ wv,
                                                               double* __restrict__ part) {
  __shared__ double red[NOALLOC_TPB];
  const int64_t g = (int64_t)blockIdx.x * NOALLOC_TPB + threadIdx.x;
  double we = 0.0;
  if (g < n) {
    const double r = rho[g], wg = w[g];
    double v0 = 0.0;
    if (r >= RHO_CUT) {
      const double c = cbrt(r);
      we = wg * (-C_X * r * c);
      v0 = wg * (-(4.0 / 3.0) * C_X * c);
    }
    wv[g] = v0;
  }
  red[threadIdx.x] = we;
  __syncthreads();
  for (int o = NOALLOC_TPB / 2; o > 0; o >>= 1) {
    if (threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
    __syncthreads();
  }
  if (threadIdx.x == 0) part[blockIdx.x] = red[0];
}

__global__ void __launch_bounds__(1024) k_sum_static(const double* __restrict__ part, int n, double* __restrict__ out) {
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

// Device address of the static array, once per device, with that device current.  In host code the array's name is a
// host-side stand-in, not a device address: the kernels get the pointer cudaGetSymbolAddress returns.
kldi_status partials_ptr(double** out) {
  static std::mutex mu;
  static double* ptr[64] = {};
  int dev = 0;
  KLDI_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) {
    set_error("kldi_xc_lda_noalloc: device index %d out of range", dev);
    return KLDI_ECUDA;
  }
  std::lock_guard<std::mutex> lock(mu);
  if (!ptr[dev]) {
    double* p = nullptr;
    KLDI_CUDA(cudaGetSymbolAddress((void**)&p, g_xc_partials));
    ptr[dev] = p;
  }
  *out = ptr[dev];
  return KLDI_OK;
}

}  // namespace
}  // namespace kldi

using namespace kldi;

extern "C" kldi_status kldi_xc_lda_noalloc(const double* rho, const double* w, int64_t n_pts, double* wv, double* Exc_dev,
                                           void* cuda_stream) {
  if (!rho || !w || !wv || !Exc_dev || n_pts <= 0) {
    set_error("kldi_xc_lda_noalloc: null argument or n_pts <= 0");
    return KLDI_EINVAL;
  }
  if (n_pts > NOALLOC_MAX_PTS) {
    set_error("kldi_xc_lda_noalloc: n_pts = %lld exceeds the static scratch of %lld points (use kldi_exc, whose plan owns "
              "its buffers)", (long long)n_pts, (long long)NOALLOC_MAX_PTS);
    return KLDI_EINVAL;
  }
  double* part = nullptr;
  kldi_status rc = partials_ptr(&part);
  if (rc != KLDI_OK) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int nb = (int)((n_pts + NOALLOC_TPB - 1) / NOALLOC_TPB);
  k_xc_lda_static<<<nb, NOALLOC_TPB, 0, st>>>(n_pts, rho, w, wv, part);
  KLDI_CUDA(cudaGetLastError());
  k_sum_static<<<1, 1024, 0, st>>>(part, nb, Exc_dev);
  KLDI_CUDA(cudaGetLastError());
  return KLDI_OK;
}

extern "C" int64_t kldi_xc_lda_noalloc_max_pts(void) { return NOALLOC_MAX_PTS; }
