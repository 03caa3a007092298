// route_noalloc.cu -- wisp_route_noalloc: the router step (a1: logits + top-k + renormalised softmax) of one layer for a small
// token batch WITHOUT any allocation, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving
// loops, harnesses that forbid it).  It is a variant of the decode path's logits kernel (decode_kernels.cuh:
// decode_logits_kernel): the same 16-column slices of the hidden state, the same fmaf chain per slice, the same 2^-32
// fixed-point int64 accumulators (decode_combine.cuh) -- but the accumulators, which the context-owning path keeps in a
// cudaMalloc'ed buffer, live here in ONE file-scope device array of fixed size:
//
//     g_route_scratch: kRouteScratchWords = 8192 int64 accumulators = 64 KiB, i.e. n_tokens * n_experts <= 8192
//     (8 tokens x 1024 experts, 64 tokens x 128 experts).  Every GPU that loads the library holds these 64 KiB until exit.
//
// In host code the array's NAME is only a host-side stand-in for the symbol, never a device address; the address is looked up
// once per device, with that device current, by cudaGetSymbolAddress (route_scratch_of) and that pointer is what the kernels get.
// All calls share the array and it keeps the last call's contents: every call clears the words it uses on its own stream first.
// Calls that overlap on the GPU (different streams, or graph replays that run concurrently) race on it -- serialise them.
#include <cstdio>
#include <mutex>

#include "common.cuh"
#include "decode_combine.cuh"
#include "router.cuh"

namespace wisp {

constexpr int kRouteScratchWords = 8192;
static __device__ __align__(256) long long g_route_scratch[kRouteScratchWords];

// Partial logits of the 16-column slices of x [T][d] for all experts, from the router weights as the caller holds them
// (row-major [E][d]): per (slice, expert) the fmaf chain of slice_logits (ascending j from 0.f), added to zfix[t][e] as a
// fixed-point integer.  Integer adds are associative, so the result does not depend on the order the CTAs arrive in.
template <typename T>
__global__ void __launch_bounds__(256) route_logits_rowmajor_kernel(const T* __restrict__ x, const T* __restrict__ w, long long* zfix,
                                                                    int n_tokens, int E, int d) {
  __shared__ float s_xn[kSliceCols];
  const int n_slices = n_tokens * (d / kSliceCols);
  for (int sl = blockIdx.x; sl < n_slices; sl += gridDim.x) {
    const int t = sl / (d / kSliceCols), j0 = (sl % (d / kSliceCols)) * kSliceCols;
    if (threadIdx.x < kSliceCols) s_xn[threadIdx.x] = to_f32<T>(x[(size_t)t * d + j0 + threadIdx.x]);
    __syncthreads();
    for (int e = threadIdx.x; e < E; e += blockDim.x) {
      const T* row = w + (size_t)e * d + j0;
      float zp = 0.f;
#pragma unroll
      for (int jj = 0; jj < kSliceCols; ++jj) zp = fmaf(to_f32<T>(row[jj]), s_xn[jj], zp);
      atomicAdd(reinterpret_cast<unsigned long long*>(zfix + (size_t)t * E + e), zfix_pack_uncounted(zp));
    }
    __syncthreads();
  }
}

// One warp per token: logits out of the accumulators (+ bias), top-k in (z desc, id asc) order, softmax over the selected k.
template <int EPL>
__global__ void __launch_bounds__(128) route_finish_kernel(const long long* __restrict__ zfix, const float* __restrict__ bias,
                                                           float* __restrict__ logits, int* __restrict__ ids, float* __restrict__ wts,
                                                           int n_tokens, int E, int k) {
  const int t = blockIdx.x * 4 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (t >= n_tokens) return;
  const long long* zt = zfix + (size_t)t * E;
  auto zf = [&](int e) { return logit_from_fix(zfix_value(zt[e]), bias ? bias[e] : 0.f); };
  topk_softmax_warp<EPL>(zf, E, k, ids + (size_t)t * k, wts + (size_t)t * k, lane);
  if (logits)
    for (int e = lane; e < E; e += 32) logits[(size_t)t * E + e] = zf(e);
}

namespace {

constexpr int kMaxDevices = 64;
std::mutex g_route_mu;
long long* g_route_ptr[kMaxDevices] = {};

// Device address of g_route_scratch on the CURRENT device, resolved once per device.
cudaError_t route_scratch_of(long long** out) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lk(g_route_mu);
  if (!g_route_ptr[dev]) {
    long long* p = nullptr;
    e = cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_route_scratch);
    if (e != cudaSuccess) return e;
    g_route_ptr[dev] = p;
  }
  *out = g_route_ptr[dev];
  return cudaSuccess;
}

}  // namespace
}  // namespace wisp

using namespace wisp;

extern "C" int wisp_route_noalloc(const void* hidden, const void* router_w, const float* router_bias, int32_t n_tokens,
                                  int32_t n_experts, int32_t d_model, int32_t top_k, int32_t dtype, float* logits, int32_t* ids,
                                  float* w, void* cuda_stream) {
  auto bad = [](const char* what) {
    std::fprintf(stderr, "wisp_route_noalloc: %s\n", what);
    return (int)WISP_EINVAL;
  };
  if (n_tokens == 0) return WISP_OK;
  if (!hidden || !router_w || !ids || !w) return bad("null hidden / router_w / ids / w");
  if (n_tokens < 0 || n_experts < 1 || n_experts > kMaxExperts || top_k < 1 || top_k > kMaxTopK || top_k > n_experts)
    return bad("n_tokens, n_experts (1..1024) or top_k (1..min(E, 32)) out of range");
  if (d_model < kSliceCols || d_model % kSliceCols) return bad("d_model must be a positive multiple of 16");
  if (dtype != WISP_F32 && dtype != WISP_BF16) return bad("dtype must be WISP_F32 or WISP_BF16");
  if ((long long)n_tokens * n_experts > kRouteScratchWords) {
    std::fprintf(stderr, "wisp_route_noalloc: n_tokens * n_experts = %lld exceeds the static scratch of %d accumulators (64 KiB)\n",
                 (long long)n_tokens * n_experts, kRouteScratchWords);
    return WISP_EINVAL;
  }
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  long long* zfix = nullptr;
  cudaError_t e = route_scratch_of(&zfix);
  if (e != cudaSuccess) {
    std::fprintf(stderr, "wisp_route_noalloc: cudaGetSymbolAddress: %s\n", cudaGetErrorString(e));
    return WISP_ECUDA;
  }
  // the array keeps the previous call's sums: clear the words this call accumulates into
  if ((e = cudaMemsetAsync(zfix, 0, (size_t)n_tokens * n_experts * sizeof(long long), st)) != cudaSuccess) {
    std::fprintf(stderr, "wisp_route_noalloc: cudaMemsetAsync: %s\n", cudaGetErrorString(e));
    return WISP_ECUDA;
  }
  const int n_slices = n_tokens * (d_model / kSliceCols);
  const int grid = n_slices < 1184 ? n_slices : 1184;
  if (dtype == WISP_F32)
    route_logits_rowmajor_kernel<float><<<grid, 256, 0, st>>>(static_cast<const float*>(hidden), static_cast<const float*>(router_w), zfix,
                                                             n_tokens, n_experts, d_model);
  else
    route_logits_rowmajor_kernel<__nv_bfloat16><<<grid, 256, 0, st>>>(static_cast<const __nv_bfloat16*>(hidden),
                                                                     static_cast<const __nv_bfloat16*>(router_w), zfix, n_tokens,
                                                                     n_experts, d_model);
  if (n_experts <= 256)
    route_finish_kernel<8><<<(n_tokens + 3) / 4, 128, 0, st>>>(zfix, router_bias, logits, ids, w, n_tokens, n_experts, top_k);
  else
    route_finish_kernel<kMaxExperts / 32><<<(n_tokens + 3) / 4, 128, 0, st>>>(zfix, router_bias, logits, ids, w, n_tokens, n_experts, top_k);
  if ((e = cudaGetLastError()) != cudaSuccess) {
    std::fprintf(stderr, "wisp_route_noalloc: launch: %s\n", cudaGetErrorString(e));
    return WISP_ECUDA;
  }
  return WISP_OK;
}
