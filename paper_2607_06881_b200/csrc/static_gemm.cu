// static_gemm.cu -- md_gemm_static: the whole path a1-a4 (include/mdgemm.h: md_gemm) for callers that can not
// allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  md_gemm needs a caller-owned
// workspace (exponent vectors, packed quarter planes, stream-K scratch); here that workspace is a FILE-SCOPE device array of
// MD_STATIC_SCRATCH_BYTES, so the call allocates nothing -- no cudaMalloc, no cudaFree, no allocating library routine -- and
// runs exactly the kernels md_gemm runs (gemm_impl), on pointers carved out of the array.
//
// What that costs and what to know:
//   * every GPU on which the library's module is loaded holds the array (64 MiB) until the process exits;
//   * the problem must fit: md_gemm_static_bytes(m, n, k, limbs) <= MD_STATIC_SCRATCH_BYTES (default options: cubes up to 496^3
//     for double double, 352^3 quad double, 192^3 octo double; hexa double never fits), otherwise MD_ERR_STATIC_LIMIT and nothing
//     is enqueued;
//   * ALL calls on a device share the one array, which keeps the previous call's contents: what must start at zero (the status
//     word here; the column maxima and stream-K counters inside the launchers) is cleared on the stream by every call, and two
//     calls that overlap on the GPU (different streams without an ordering between them) RACE -- serialise them;
//   * in HOST code the array's name is a host-side stand-in, not a device address: the address is taken once per device with
//     cudaGetSymbolAddress, with that device current, in this file.
#include "api_internal.h"

namespace {

constexpr size_t MD_STATIC_SCRATCH_BYTES = (size_t)64 << 20;
static __device__ __align__(256) unsigned char md_static_scratch[MD_STATIC_SCRATCH_BYTES];

// device address of the array on each device (0 = not asked yet); the current device's entry is filled on first use
void* g_static_ptr[md::MD_MAX_DEVICES] = {};

// returns nullptr (and leaves *err set) when the address can not be obtained
void* static_scratch_ptr(cudaError_t* err) {
  const int dev = md::current_device();
  if (dev < 0 || dev >= md::MD_MAX_DEVICES) {
    *err = cudaErrorInvalidDevice;
    return nullptr;
  }
  if (!g_static_ptr[dev]) {
    void* p = nullptr;
    *err = cudaGetSymbolAddress(&p, md_static_scratch);  // the current device's copy of the array
    if (*err != cudaSuccess || !p) return nullptr;
    g_static_ptr[dev] = p;
  }
  *err = cudaSuccess;
  return g_static_ptr[dev];
}

// bytes of the array a problem uses with the current options: the layout gemm_impl carves for the kernel it will pick
size_t static_need(int m, int n, int k, int limbs) {
  const int Q = md::quarters_for(limbs), S = md::orders_for(limbs);
  const md::KernelPick pick = md::pick_kernel(m, n, k, limbs, Q, S, md::slice_bits(), false, true);
  if (pick.family == md::GEMM_NONE) return 0;
  return md::carve(nullptr, m, n, k, Q, S, pick).total;
}

}  // namespace

extern "C" {

size_t md_static_scratch_bytes(void) { return MD_STATIC_SCRATCH_BYTES; }

size_t md_gemm_static_bytes(int m, int n, int k, int limbs) {
  if (m <= 0 || n <= 0 || k <= 0 || !(limbs == 2 || limbs == 4 || limbs == 8 || limbs == 16)) return 0;
  return static_need(m, n, k, limbs);
}

md_status md_gemm_static(int m, int n, int k, int limbs, const double* A_planes, const double* B_planes, double* C_planes,
                         md_stream stream) {
  const md_status st = md::check_gemm_args(m, n, k, limbs, A_planes, B_planes, C_planes, false);
  if (st != MD_OK) return st;
  const size_t need = static_need(m, n, k, limbs);
  if (need == 0) return MD_ERR_UNSUPPORTED;
  if (need > MD_STATIC_SCRATCH_BYTES) return MD_ERR_STATIC_LIMIT;  // nothing has been enqueued
  cudaError_t err;
  void* ws = static_scratch_ptr(&err);
  if (!ws) return MD_ERR_CUDA;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  // the array keeps the previous call's contents: the status word of THIS call starts at zero
  if (cudaMemsetAsync(ws, 0, md::WS_ALIGN, s) != cudaSuccess) return MD_ERR_CUDA;
  return md::gemm_impl(m, n, k, limbs, md::quarters_for(limbs), md::orders_for(limbs), A_planes, B_planes, C_planes, nullptr, ws,
                       MD_STATIC_SCRATCH_BYTES, s, true);
}

md_status md_gemm_static_read_flags(uint32_t* flags_host, md_stream stream) {
  if (!flags_host) return MD_ERR_BAD_ARG;
  cudaError_t err;
  void* ws = static_scratch_ptr(&err);
  if (!ws) return MD_ERR_CUDA;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  if (cudaMemcpyAsync(flags_host, ws, sizeof(uint32_t), cudaMemcpyDeviceToHost, s) != cudaSuccess) return MD_ERR_CUDA;
  return cudaStreamSynchronize(s) == cudaSuccess ? MD_OK : MD_ERR_CUDA;
}

}  // extern "C"
