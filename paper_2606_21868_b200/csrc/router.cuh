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

// Top-k + softmax of n_tokens rows of logits held in shared memory (z [n_tokens][E], read only), by `nthr` threads
// (threadIdx.x < nthr) that synchronise through named barrier `bar`.  Selection by rank counting, which IS the
// definition (G7): rank(e) = #{j : z_j > z_e or (z_j == z_e and j < e)}; the experts of rank < k are the top-k in
// (z desc, id asc) order.  w_i = exp(z_i - z_0) / sum_j exp(z_j - z_0), the sum taken in rank order j = 0..k-1.
// ids_out / w_out: [n_tokens][k] (any address space); selz: [n_tokens][k] floats of shared scratch.
__device__ __forceinline__ void topk_softmax_block(const float* z, int n_tokens, int E, int k, int* ids_out, float* w_out,
                                                   float* selz, int nthr, int bar) {
  const int tid = threadIdx.x;
  for (int idx = tid; idx < n_tokens * E; idx += nthr) {
    const int t = idx / E, e = idx % E;
    const float* row = z + (size_t)t * E;
    const float ze = row[e];
    int rank = 0;
    if ((E & 3) == 0 && (((size_t)row) & 15) == 0) {       // all lanes read the same address: shared-memory broadcast
      const float4* row4 = reinterpret_cast<const float4*>(row);
#pragma unroll 4
      for (int j4 = 0; j4 < E / 4; ++j4) {
        const float4 v = row4[j4];
        const int j = j4 * 4;
        rank += (v.x > ze) || (v.x == ze && j < e);
        rank += (v.y > ze) || (v.y == ze && j + 1 < e);
        rank += (v.z > ze) || (v.z == ze && j + 2 < e);
        rank += (v.w > ze) || (v.w == ze && j + 3 < e);
      }
    } else {
      for (int j = 0; j < E; ++j) {
        const float zj = row[j];
        rank += (zj > ze) || (zj == ze && j < e);
      }
    }
    if (rank < k) { ids_out[t * k + rank] = e; selz[t * k + rank] = ze; }
  }
  asm volatile("bar.sync %0, %1;" ::"r"(bar), "r"(nthr) : "memory");
  for (int idx = tid; idx < n_tokens * k; idx += nthr) {
    const int t = idx / k;
    const float z0 = selz[t * k];
    float den = 0.f;
    for (int j = 0; j < k; ++j) den += expf(selz[t * k + j] - z0);   // fixed order
    w_out[idx] = expf(selz[idx] - z0) / den;
  }
  asm volatile("bar.sync %0, %1;" ::"r"(bar), "r"(nthr) : "memory");
}

// 4 tokens per block of 128 threads.  smem: 4 * E floats (logits) + 4 * k floats.
__global__ void __launch_bounds__(128) topk_softmax_kernel(const float* __restrict__ z, int* __restrict__ ids,
                                                           float* __restrict__ w, int n_tokens, int E, int k) {
  extern __shared__ float sz[];
  const int t0 = blockIdx.x * 4, nt = min(4, n_tokens - t0);
  for (int i = threadIdx.x; i < nt * E; i += 128) sz[i] = z[(size_t)t0 * E + i];
  __syncthreads();
  topk_softmax_block(sz, nt, E, k, ids + (size_t)t0 * k, w + (size_t)t0 * k, sz + 4 * E, 128, 0);
}

}  // namespace wisp
