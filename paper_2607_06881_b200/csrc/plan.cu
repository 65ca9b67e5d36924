// plan.cu -- kernels of md_plan_quarters (include/mdgemm.h; R15): how far below 2^(E_i + F_j) the entries of
// |A||B| fall, which decides how many quarters the common-exponent grid of a row / column needs (R5).
#include <limits.h>

#include "md_common.cuh"
#include "md_kernels.h"

namespace md {
namespace {

__global__ void __launch_bounds__(256) abs_kernel(size_t count, const double* __restrict__ in, double* __restrict__ out) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < count; i += (size_t)gridDim.x * blockDim.x)
    out[i] = fabs(in[i]);
}

// D = max over (i, j) with W_ij > 0 of E_i + F_j - ilogb(W_ij); one row per blockIdx.y, columns strided over the block.
__global__ void __launch_bounds__(256) spread_kernel(int m, int n, const double* __restrict__ W,
                                                     const int32_t* __restrict__ expA, const int32_t* __restrict__ expB,
                                                     int32_t* spread) {
  int best = INT_MIN;
  for (int i = blockIdx.x; i < m; i += gridDim.x) {
    const int Ei = expA[i];
    for (int j = threadIdx.x; j < n; j += blockDim.x) {
      const double w = W[(size_t)i * n + j];
      if (w > 0.0) {
        const int e = (int)((__double_as_longlong(w) >> 52) & 0x7ff) - 1023;  // ilogb of a normal double
        best = max(best, Ei + expB[j] - e);
      }
    }
  }
  best = __reduce_max_sync(0xffffffffu, best);
  if ((threadIdx.x & 31) == 0 && best != INT_MIN) atomicMax(spread, best);
}

}  // namespace

cudaError_t launch_abs(size_t count, const double* in, double* out, cudaStream_t stream, uint64_t* launches) {
  const size_t want = (count + 255) / 256;
  const int cap = (sm_count() > 0 ? sm_count() : 1) * 32;
  abs_kernel<<<(unsigned)(want < (size_t)cap ? want : (size_t)cap), 256, 0, stream>>>(count, in, out);
  *launches += 1;
  return cudaGetLastError();
}

cudaError_t launch_spread(int m, int n, const double* W, const int32_t* expA, const int32_t* expB, int32_t* spread,
                          cudaStream_t stream, uint64_t* launches) {
  const int cap = (sm_count() > 0 ? sm_count() : 1) * 16;
  spread_kernel<<<m < cap ? m : cap, 256, 0, stream>>>(m, n, W, expA, expB, spread);
  *launches += 1;
  return cudaGetLastError();
}

}  // namespace md
