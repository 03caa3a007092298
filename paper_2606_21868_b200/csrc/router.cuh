// router.cuh -- (a1) router GEMV + top-k + softmax over the selected logits.
// The paper does not define the router (it is the engine's); BASELINE.json does:
// "top-k routing with renormalised softmax over the top-k" (G7): z_e = bias_e + <W_r[e], x>,
// ids = k largest by (z desc, id asc), w_i = exp(z_i - z_0) / sum_j exp(z_j - z_0).
#pragma once
#include "common.cuh"

namespace wisp {

constexpr int kRouterTokTile = 4;

// One warp: logits of expert row `wrow` against tokens t0 .. t0+nt-1 (nt <= 4) of x.  Canonical order (common.cuh):
// lane l takes the 16-byte chunks l, l+32, ... in ascending order into one fp32 accumulator per token, then the
// xor butterfly; lane 0 writes z[t][e] = sum + bias.  Used by the standalone kernel and the persistent decode kernel.
template <typename T>
__device__ __forceinline__ void router_row_warp(const T* x, const T* wrow, float bias_e, float* z, int e, int t0, int nt,
                                                int E, int d, int lane) {
  constexpr int N = Chunk<T>::N;
  constexpr int UN = 8;                       // weight chunks in flight per lane (loads hoisted; the FMA order is unchanged)
  float acc[kRouterTokTile] = {0.f, 0.f, 0.f, 0.f};
  for (int c0 = lane * N; c0 < d; c0 += UN * 32 * N) {
    uint4 raw[UN];
#pragma unroll
    for (int u = 0; u < UN; ++u) {
      const int c = c0 + u * 32 * N;
      if (c < d) raw[u] = *reinterpret_cast<const uint4*>(wrow + c);
    }
#pragma unroll
    for (int u = 0; u < UN; ++u) {
      const int c = c0 + u * 32 * N;
      if (c < d) {
        float wv[N];
        ChunkW<T>::widen(raw[u], wv);
#pragma unroll
        for (int tt = 0; tt < kRouterTokTile; ++tt) {
          if (tt < nt) {
            float xv[N];
            Chunk<T>::load(x + (size_t)(t0 + tt) * d + c, xv);
#pragma unroll
            for (int j = 0; j < N; ++j) acc[tt] = fmaf(wv[j], xv[j], acc[tt]);
          }
        }
      }
    }
  }
#pragma unroll
  for (int tt = 0; tt < kRouterTokTile; ++tt) {
    float s = warp_sum(acc[tt]);
    if (tt < nt && lane == 0) z[(size_t)(t0 + tt) * E + e] = s + bias_e;
  }
}

// grid (ceil(E/8), ceil(T/4)), block 256: warp = one expert row against up to 4 tokens.
template <typename T>
__global__ void __launch_bounds__(256) router_logits_kernel(const T* __restrict__ x, const T* __restrict__ w_r,
                                                            const float* __restrict__ bias, float* __restrict__ z,
                                                            int n_tokens, int E, int d) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int e = blockIdx.x * 8 + warp;
  const int t0 = blockIdx.y * kRouterTokTile;
  if (e >= E) return;
  router_row_warp<T>(x, w_r + (size_t)e * d, bias ? bias[e] : 0.f, z, e, t0, min(kRouterTokTile, n_tokens - t0), E, d, lane);
}

// Top-k + softmax of ONE token's logits by ONE warp ("warp-shuffle softmax and top-k", BASELINE.json north_star; G7).
// Lane l owns the logits of experts l, l+32, ... as order-preserving 32-bit keys.  One round = the warp maximum of the keys
// (redux.sync.max), then the LOWEST expert id among the lanes that hold that maximum (redux.sync.min): the largest logit
// with ties going to the lower id; k rounds give ids in (z desc, id asc) order.  -0 compares equal to +0 and a NaN ranks
// with -inf (it can never corrupt an id: every selected id is a real expert).
// w_i = exp(z_i - z_0) / sum_j exp(z_j - z_0), the sum taken in rank order j = 0..k-1 (every lane computes the same chain).
// EPL = logits per lane (E <= 32 * EPL); zf(e) returns the logit of expert e.  ids_out / w_out: [k].
__device__ __forceinline__ unsigned topk_key(float z) {
  z += 0.0f;                                            // -0 -> +0
  unsigned u = __float_as_uint(z);
  if (z != z) u = 0xff800000u;                          // NaN -> -inf
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);    // unsigned order == float order; every key is > 0
}
__device__ __forceinline__ float topk_key_logit(unsigned u) {
  u = (u & 0x80000000u) ? (u & 0x7fffffffu) : ~u;
  return __uint_as_float(u);
}
template <int EPL, typename ZF>
__device__ __forceinline__ void topk_softmax_warp(ZF zf, int E, int k, int* ids_out, float* w_out, int lane) {
  unsigned key[EPL];
#pragma unroll
  for (int j = 0; j < EPL; ++j) {
    const int e = lane + 32 * j;
    key[j] = e < E ? topk_key(zf(e)) : 0u;               // 0 = absent / already taken
  }
  float my_z = 0.f;                                     // lane r keeps the logit of rank r
  for (int r = 0; r < k; ++r) {
    unsigned best = 0u;
    int best_j = 0;
#pragma unroll
    for (int j = EPL - 1; j >= 0; --j)                   // descending j with >= : among equal keys the lowest id of the lane wins
      if (key[j] >= best) { best = key[j]; best_j = j; }
    const unsigned top = __reduce_max_sync(0xffffffffu, best);
    const unsigned e = __reduce_min_sync(0xffffffffu, best == top ? (unsigned)(lane + 32 * best_j) : 0xffffffffu);
#pragma unroll
    for (int j = 0; j < EPL; ++j)
      if ((int)e == lane + 32 * j) key[j] = 0u;
    if (lane == r) { my_z = topk_key_logit(top); ids_out[r] = (int)e; }
  }
  const float z0 = __shfl_sync(0xffffffffu, my_z, 0);
  float den = 0.f;
  for (int j = 0; j < k; ++j) den += expf(__shfl_sync(0xffffffffu, my_z, j) - z0);   // fixed order
  if (lane < k) w_out[lane] = expf(my_z - z0) / den;
}

// Prefill / multi-kernel path: one warp per token, 4 tokens per block of 128 threads; z [n_tokens][E] in global memory.
template <int EPL>
__global__ void __launch_bounds__(128) topk_softmax_kernel(const float* __restrict__ z, int* __restrict__ ids,
                                                           float* __restrict__ w, int n_tokens, int E, int k) {
  const int t = blockIdx.x * 4 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (t >= n_tokens) return;
  const float* row = z + (size_t)t * E;
  topk_softmax_warp<EPL>([&](int e) { return row[e]; }, E, k, ids + (size_t)t * k, w + (size_t)t * k, lane);
}

}  // namespace wisp
