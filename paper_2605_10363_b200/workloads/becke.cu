// Becke fuzzy-cell partition factors for the synthetic workload generator (inputs only).
// Same formula as generate._becke_numpy: P_A = prod_{B!=A} s(mu_AB), mu_AB=(r_A-r_B)/R_AB,
// f <- 1.5 f - 0.5 f^3 three times, s=(1-f)/2; result = P_owner / sum_B P_B.
// Not part of the KerneLDI hot path and not linked into libkldi.so.
#include <cuda_runtime.h>
#include <cstdint>

namespace {
__global__ void becke_kernel(const double* __restrict__ atoms, const double* __restrict__ inv_r,
                             const double* __restrict__ pts, const int* __restrict__ owner,
                             double* __restrict__ out, long long n_pts, int n_at) {
  extern __shared__ double sh[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
  double* d = sh + (size_t)warp * n_at;
  for (long long g = (long long)blockIdx.x * nwarp + warp; g < n_pts; g += (long long)gridDim.x * nwarp) {
    const double x = pts[3 * g], y = pts[3 * g + 1], z = pts[3 * g + 2];
    for (int b = lane; b < n_at; b += 32) {
      const double dx = x - atoms[3 * b], dy = y - atoms[3 * b + 1], dz = z - atoms[3 * b + 2];
      d[b] = sqrt(dx * dx + dy * dy + dz * dz);
    }
    __syncwarp();
    const int own = owner[g];
    double tot = 0.0, pown = 0.0;
    for (int a = lane; a < n_at; a += 32) {
      const double da = d[a];
      double p = 1.0;
      for (int b = 0; b < n_at; ++b) {
        if (b == a) continue;
        double f = (da - d[b]) * inv_r[(size_t)b * n_at + a];
        f = 1.5 * f - 0.5 * f * f * f;
        f = 1.5 * f - 0.5 * f * f * f;
        f = 1.5 * f - 0.5 * f * f * f;
        p *= 0.5 * (1.0 - f);
      }
      tot += p;
      if (a == own) pown = p;
    }
    for (int o = 16; o > 0; o >>= 1) {
      tot += __shfl_xor_sync(0xffffffffu, tot, o);
      pown += __shfl_xor_sync(0xffffffffu, pown, o);
    }
    if (lane == 0) out[g] = pown / tot;
    __syncwarp();
  }
}
}  // namespace

// all pointers are DEVICE pointers; inv_r is the [n_at][n_at] matrix of 1/R_AB (diagonal unused)
extern "C" int wl_becke_partition(const double* atoms, const double* inv_r, const double* pts,
                                  const int* owner, double* out, long long n_pts, int n_at, void* stream) {
  int warps = 8;
  while (warps > 1 && (size_t)warps * n_at * sizeof(double) > 200 * 1024) warps >>= 1;
  size_t smem = (size_t)warps * n_at * sizeof(double);
  if (smem > 200 * 1024) return -1;
  cudaFuncSetAttribute(becke_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  int dev = 0, nsm = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
  int blocks = nsm * (smem > 100 * 1024 ? 1 : 2);
  becke_kernel<<<blocks, warps * 32, smem, (cudaStream_t)stream>>>(atoms, inv_r, pts, owner, out, n_pts, n_at);
  return cudaGetLastError() == cudaSuccess ? 0 : -2;
}
