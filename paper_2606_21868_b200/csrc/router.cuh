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
  float acc[kRouterTokTile] = {0.f, 0.f, 0.f, 0.f};
  for (int c = lane * N; c < d; c += 32 * N) {
    float wv[N];
    Chunk<T>::load(wrow + c, wv);
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

// One warp, one token: `row` = that token's E logits in shared memory (destroyed).  ids (z desc, id asc) and the
// softmax over the selected k (G7) go to ids_out[0..k) / w_out[0..k) (any address space).
__device__ __forceinline__ void topk_softmax_warp(float* row, int E, int k, int lane, int* ids_out, float* w_out) {
  float my_z = 0.f;  // lane i keeps the i-th selected logit
  int my_id = 0;
  for (int i = 0; i < k; ++i) {
    float bz = -INFINITY;
    int be = 0x7fffffff;
    for (int e = lane; e < E; e += 32) {     // ascending e within a lane: first max wins -> lower id
      float v = row[e];
      if (v > bz) { bz = v; be = e; }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      float oz = __shfl_xor_sync(0xffffffffu, bz, o);
      int oe = __shfl_xor_sync(0xffffffffu, be, o);
      if (oz > bz || (oz == bz && oe < be)) { bz = oz; be = oe; }
    }
    if (lane == i) { my_z = bz; my_id = be; }
    if (lane == 0) row[be] = -INFINITY;
    __syncwarp();
  }
  const float z0 = __shfl_sync(0xffffffffu, my_z, 0);
  const float ex = (lane < k) ? expf(my_z - z0) : 0.f;
  float den = 0.f;
  for (int i = 0; i < k; ++i) den += __shfl_sync(0xffffffffu, ex, i);   // fixed order
  if (lane < k) {
    ids_out[lane] = my_id;
    w_out[lane] = ex / den;
  }
}

// One warp per token; block 128 = 4 tokens.  smem: 4 * E floats.
__global__ void __launch_bounds__(128) topk_softmax_kernel(const float* __restrict__ z, int* __restrict__ ids,
                                                           float* __restrict__ w, int n_tokens, int E, int k) {
  extern __shared__ float sz[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int t = blockIdx.x * 4 + warp;
  if (t >= n_tokens) return;
  float* row = sz + warp * E;
  for (int e = lane; e < E; e += 32) row[e] = z[(size_t)t * E + e];
  __syncwarp();
  topk_softmax_warp(row, E, k, lane, ids + (size_t)t * k, w + (size_t)t * k);
}

}  // namespace wisp
