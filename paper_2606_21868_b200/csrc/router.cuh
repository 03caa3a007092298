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
// Lane l owns the experts l, l+32, ... (coalesced logit reads) as order-preserving 32-bit keys.  One round = the warp maximum of
// the lanes' best keys (redux.sync.max); if one lane holds it (ballot) that is the winner, and on a tie the LOWEST expert id
// among the tied lanes wins (redux.sync.min, rare): the largest logit with ties going to the lower id; k rounds give ids in
// (z desc, id asc) order.  -0 compares equal to +0 and a NaN ranks with -inf (it can never corrupt an id: every selected id
// is a real expert).
// w_i = exp(z_i - z_0) / sum_j exp(z_j - z_0), the sum taken in rank order j = 0..k-1.
// EPL = compile-time bound of per (E <= 32 * EPL); zf(e) returns the logit of expert e.  ids_out / w_out: [k], shared or global;
// w_out doubles as scratch for the selected logits.
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
  for (int r = 0; r < k; ++r) {
    unsigned best = 0u;
    int best_j = 0;
#pragma unroll
    for (int j = EPL - 1; j >= 0; --j)                   // descending j with >= : among equal keys the lane's lowest id wins
      if (key[j] >= best) { best = key[j]; best_j = j; }
    const unsigned top = __reduce_max_sync(0xffffffffu, best);
    const unsigned tied = __ballot_sync(0xffffffffu, best == top);
    int e = lane + 32 * best_j;
    if (tied & (tied - 1u)) e = (int)__reduce_min_sync(0xffffffffu, best == top ? (unsigned)e : 0xffffffffu);   // several lanes: lowest id
    else e = __shfl_sync(0xffffffffu, e, __ffs(tied) - 1);
    if ((e & 31) == lane) {
      ids_out[r] = e;
      w_out[r] = topk_key_logit(top);
#pragma unroll
      for (int j = 0; j < EPL; ++j)
        if (j == (e >> 5)) key[j] = 0u;
    }
  }
  __syncwarp();
  const float z0 = w_out[0];
  const float ex = lane < k ? expf(w_out[lane] - z0) : 0.f;
  float den = 0.f;
  for (int j = 0; j < k; ++j) den += __shfl_sync(0xffffffffu, ex, j);   // fixed order
  __syncwarp();
  if (lane < k) w_out[lane] = ex / den;
}

// The same selection by a whole thread block (the fused decode kernel: 256 threads, 1..8 tokens): rank counting, which IS the
// definition (G7): rank(e) = #{j : z_j > z_e or (z_j == z_e and j < e)} on the same 32-bit keys; the experts of rank < k are
// the top-k in (z desc, id asc) order.  One pass of independent compares instead of k dependent warp reductions.  The softmax
// is the same chain as in topk_softmax_warp, so both give the same ids and the same weight bits.
// zf(t, e) returns the logit; keys: n_tokens * E words of shared scratch; threads tid < nthr synchronise on named barrier `bar`.
template <typename ZF>
__device__ __forceinline__ void topk_softmax_block(ZF zf, int n_tokens, int E, int k, int* ids_out, float* w_out, unsigned* keys, int tid,
                                                   int nthr, int bar) {
  for (int idx = tid; idx < n_tokens * E; idx += nthr) keys[idx] = topk_key(zf(idx / E, idx % E));
  asm volatile("bar.sync %0, %1;" ::"r"(bar), "r"(nthr) : "memory");
  for (int idx = tid; idx < n_tokens * E; idx += nthr) {
    const int t = idx / E, e = idx % E;
    const unsigned* row = keys + (size_t)t * E;
    const unsigned me = row[e];
    int rank = 0;
    if ((E & 3) == 0 && (((size_t)row) & 15) == 0) {       // all lanes of a token read the same address: shared-memory broadcast
      const uint4* row4 = reinterpret_cast<const uint4*>(row);
#pragma unroll 4
      for (int j4 = 0; j4 < E / 4; ++j4) {
        const uint4 v = row4[j4];
        const int j = j4 * 4;
        rank += (v.x > me) || (v.x == me && j < e);
        rank += (v.y > me) || (v.y == me && j + 1 < e);
        rank += (v.z > me) || (v.z == me && j + 2 < e);
        rank += (v.w > me) || (v.w == me && j + 3 < e);
      }
    } else {
      for (int j = 0; j < E; ++j) rank += (row[j] > me) || (row[j] == me && j < e);
    }
    if (rank < k) { ids_out[t * k + rank] = e; w_out[t * k + rank] = topk_key_logit(me); }
  }
  asm volatile("bar.sync %0, %1;" ::"r"(bar), "r"(nthr) : "memory");
  float val = 0.f;
  const bool mine = tid < n_tokens * k;
  if (mine) {
    const int t = tid / k;
    const float z0 = w_out[t * k];
    float den = 0.f;
    for (int j = 0; j < k; ++j) den += expf(w_out[t * k + j] - z0);   // fixed order
    val = expf(w_out[tid] - z0) / den;
  }
  asm volatile("bar.sync %0, %1;" ::"r"(bar), "r"(nthr) : "memory");
  if (mine) w_out[tid] = val;
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
