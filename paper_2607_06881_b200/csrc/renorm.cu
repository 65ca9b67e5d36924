// renorm.cu -- step a4 as a standalone kernel (include/mdgemm.h: md_renorm): the `orders` order matrices C^(s) are summed,
// error free, into `limbs` limb planes.  Same device function as the fused epilogue of qgemm.cu.
// HBM-bound: reads 8*orders and writes 8*limbs bytes per element.
#include "md_common.cuh"
#include "md_kernels.h"

namespace md {
namespace {

template <int L>
__global__ void __launch_bounds__(256) renorm_kernel(size_t total, int S, const double* __restrict__ order_planes,
                                                     double* __restrict__ C_planes) {
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= total) return;
  double r[L + 1], out[L];
#pragma unroll
  for (int l = 0; l <= L; l++) r[l] = 0.0;
  // smallest order first (R9); 4 loads in flight per thread
  int s = S - 1;
  for (; s >= 3; s -= 4) {
    double x[4];
#pragma unroll
    for (int u = 0; u < 4; u++) x[u] = order_planes[(size_t)(s - u) * total + idx];
#pragma unroll
    for (int u = 0; u < 4; u++) renorm_add<L>(r, x[u]);
  }
  for (; s >= 0; s--) renorm_add<L>(r, order_planes[(size_t)s * total + idx]);
  renorm_finish<L>(r, out);
#pragma unroll
  for (int l = 0; l < L; l++) C_planes[(size_t)l * total + idx] = out[l];
}

template <int L>
cudaError_t dispatch_orders(int S, size_t total, const double* in, double* out, cudaStream_t stream) {
  const unsigned blocks = (unsigned)((total + 255) / 256);
  renorm_kernel<L><<<blocks, 256, 0, stream>>>(total, S, in, out);
  return cudaGetLastError();
}

}  // namespace

cudaError_t launch_renorm(int m, int n, int limbs, int orders, const double* order_planes, double* C_planes,
                          cudaStream_t stream, uint64_t* launches) {
  const size_t total = (size_t)m * n;
  cudaError_t err;
  switch (limbs) {
    case 1: err = dispatch_orders<1>(orders, total, order_planes, C_planes, stream); break;
    case 2: err = dispatch_orders<2>(orders, total, order_planes, C_planes, stream); break;
    case 4: err = dispatch_orders<4>(orders, total, order_planes, C_planes, stream); break;
    case 8: err = dispatch_orders<8>(orders, total, order_planes, C_planes, stream); break;
    case 16: err = dispatch_orders<16>(orders, total, order_planes, C_planes, stream); break;
    default: return cudaErrorInvalidValue;
  }
  if (err == cudaSuccess) *launches += 1;
  return err;
}

}  // namespace md
