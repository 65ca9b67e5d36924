// probe.cu -- calibration kernel behind md_probe_dmma (include/mdgemm.h): the FP64 tensor (DMMA) peak of the device this
// library runs on, i.e. the denominator of the roofline of the fused quarter GEMM.  Not a step of
// the hot path and not used by it.
//
// Every warp keeps ACC independent 8x8 accumulator tiles in registers and issues mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4)
// back to back on register operands: no shared memory, no global loads, nothing but the tensor pipe.  The operands are
// 13-bit integers (the magnitude of the quarters the real kernel multiplies), so that data-dependent power draw is
// comparable; the accumulators stay exact (iters * 4 * 2^26 < 2^53 for iters < 2^25).
#include "md_common.cuh"
#include "md_kernels.h"

namespace md {
namespace {

constexpr int PROBE_ACC = 8;

__global__ void __launch_bounds__(1024, 1) dmma_probe_kernel(int iters, double* __restrict__ sink) {
  const int lane = threadIdx.x & 31;
  double c[PROBE_ACC][2];
#pragma unroll
  for (int j = 0; j < PROBE_ACC; j++) c[j][0] = c[j][1] = 0.0;
  double a = (double)((lane * 2654435761u + blockIdx.x * 40503u) % 8191u) - 4095.0;
  double b = (double)((threadIdx.x * 2246822519u + 12345u) % 8191u) - 4095.0;
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int j = 0; j < PROBE_ACC; j++)
      asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                   : "+d"(c[j][0]), "+d"(c[j][1])
                   : "d"(a), "d"(b));
  }
  double sum = 0.0;
#pragma unroll
  for (int j = 0; j < PROBE_ACC; j++) sum += c[j][0] + c[j][1];
  if (sink) sink[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = sum;
}

}  // namespace

cudaError_t launch_dmma_probe(int blocks, int warps_per_block, int iters, double* sink, cudaStream_t stream,
                              uint64_t* launches, uint64_t* flops) {
  dmma_probe_kernel<<<blocks, warps_per_block * 32, 0, stream>>>(iters, sink);
  *launches += 1;
  *flops = (uint64_t)blocks * warps_per_block * (uint64_t)iters * PROBE_ACC * 512ull;  // 2 * 8 * 8 * 4 per DMMA
  return cudaGetLastError();
}

}  // namespace md
