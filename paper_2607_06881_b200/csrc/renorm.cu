// renorm.cu -- step a4 as a standalone kernel (include/mdgemm.h: md_renorm): the `orders` order matrices C^(s) are summed,
// error free, into `limbs` limb planes.  Same device function as the fused epilogue of qgemm.cu.
// HBM-bound: reads 8*orders and writes 8*limbs bytes per element.
#include "md_common.cuh"
#include "md_kernels.h"

namespace md {
namespace {

template <int L, int S>
__global__ void __launch_bounds__(256) renorm_kernel(size_t total, const double* __restrict__ order_planes,
                                                     double* __restrict__ C_planes) {
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= total) return;
  double c[S], out[L];
#pragma unroll
  for (int s = 0; s < S; s++) c[s] = order_planes[(size_t)s * total + idx];
  renorm_orders<L, S>(c, out);
#pragma unroll
  for (int l = 0; l < L; l++) C_planes[(size_t)l * total + idx] = out[l];
}

template <int L>
cudaError_t dispatch_orders(int S, size_t total, const double* in, double* out, cudaStream_t stream) {
  const unsigned blocks = (unsigned)((total + 255) / 256);
  switch (S) {
#define MD_CASE(S_) case S_: renorm_kernel<L, S_><<<blocks, 256, 0, stream>>>(total, in, out); break;
    MD_CASE(1) MD_CASE(2) MD_CASE(3) MD_CASE(4) MD_CASE(5) MD_CASE(6) MD_CASE(7) MD_CASE(8) MD_CASE(9) MD_CASE(10)
    MD_CASE(11) MD_CASE(12) MD_CASE(13) MD_CASE(14) MD_CASE(15) MD_CASE(16) MD_CASE(17) MD_CASE(18) MD_CASE(19)
    MD_CASE(20) MD_CASE(21) MD_CASE(22) MD_CASE(23) MD_CASE(24)
#undef MD_CASE
    default: return cudaErrorInvalidValue;
  }
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
    default: return cudaErrorInvalidValue;
  }
  if (err == cudaSuccess) *launches += 1;
  return err;
}

}  // namespace md
