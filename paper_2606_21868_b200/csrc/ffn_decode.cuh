// ffn_decode.cuh -- (a4) decode expert SwiGLU FFN over slot-indirected weights + weighted combine, as
// memory-bound GEMV kernels (1 flop/byte: plain ALUs, no tensor cores).
//   g = W_gate[s] x_t, u = W_up[s] x_t, a = silu(g) * u   (gate_up kernel, a kept in fp32)
//   y = W_down[s] a                                           (down kernel, y staged in fp32 per (token, rank))
//   out_t = sum_{i<k} w[t,i] * y_{t,i}  in rank order         (combine kernel)
// The FFN itself is the engine's in the paper ("unmodified fused-MoE kernel");
// BASELINE.json fixes SwiGLU (G8, G21).
#pragma once
#include "common.cuh"

namespace wisp {

constexpr int kFfnThreads = 256;     // 8 warps; one warp = one weight row (pair of rows for gate/up)

__device__ __forceinline__ float silu_f(float v) { return v / (1.0f + expf(-v)); }

// Work item = (entry i of the wave, row r < d_ff); warps take items round-robin over the whole grid.
template <typename T>
__global__ void __launch_bounds__(kFfnThreads) decode_gate_up_kernel(PlanPtrs plan, int wave, int C,
                                                                     const T* __restrict__ pool, size_t blob_elems,
                                                                     int L, int layer, const T* __restrict__ x,
                                                                     float* __restrict__ act, int d, int d_ff, int k) {
  constexpr int N = Chunk<T>::N;
  if (wave >= plan.hdr[0]) return;
  const int lo = wave * C, nw = min(plan.hdr[1], lo + C) - lo;
  const int lane = threadIdx.x & 31;
  const int gw = (blockIdx.x * kFfnThreads + threadIdx.x) >> 5;
  const int n_warps = (gridDim.x * kFfnThreads) >> 5;
  const size_t gu = (size_t)d_ff * d;
  for (int item = gw; item < nw * d_ff; item += n_warps) {
    const int i = lo + item / d_ff, r = item % d_ff;
    const int e = plan.entry_expert[i];
    const T* wg = pool + ((size_t)plan.entry_slot[i] * L + layer) * blob_elems + (size_t)r * d;
    const T* wu = wg + gu;
    const int cnt = plan.exp_count[e];
    const int* pl = plan.pair_list + plan.exp_offset[e];
    for (int p0 = 0; p0 < cnt; p0 += 4) {
      const int np = min(4, cnt - p0);
      int pr[4];
      float ag[4] = {0.f, 0.f, 0.f, 0.f}, au[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
      for (int q = 0; q < 4; ++q) pr[q] = q < np ? pl[p0 + q] : 0;
      for (int c = lane * N; c < d; c += 32 * N) {
        float gv[N], uv[N];
        Chunk<T>::load_stream(wg + c, gv);
        Chunk<T>::load_stream(wu + c, uv);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          if (q < np) {
            float xv[N];
            Chunk<T>::load(x + (size_t)(pr[q] / k) * d + c, xv);
#pragma unroll
            for (int j = 0; j < N; ++j) { ag[q] = fmaf(gv[j], xv[j], ag[q]); au[q] = fmaf(uv[j], xv[j], au[q]); }
          }
        }
      }
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const float g = warp_sum(ag[q]), u = warp_sum(au[q]);
        if (q < np && lane == 0) act[(size_t)pr[q] * d_ff + r] = silu_f(g) * u;
      }
    }
  }
}

// Work item = (entry i, output row j < d): y[pair, j] = <W_down[j, :], a[pair, :]>.
template <typename T>
__global__ void __launch_bounds__(kFfnThreads) decode_down_kernel(PlanPtrs plan, int wave, int C,
                                                                  const T* __restrict__ pool, size_t blob_elems, int L,
                                                                  int layer, const float* __restrict__ act,
                                                                  float* __restrict__ ystage, int d, int d_ff) {
  constexpr int N = Chunk<T>::N;
  if (wave >= plan.hdr[0]) return;
  const int lo = wave * C, nw = min(plan.hdr[1], lo + C) - lo;
  const int lane = threadIdx.x & 31;
  const int gw = (blockIdx.x * kFfnThreads + threadIdx.x) >> 5;
  const int n_warps = (gridDim.x * kFfnThreads) >> 5;
  const size_t gu2 = 2 * (size_t)d_ff * d;
  for (int item = gw; item < nw * d; item += n_warps) {
    const int i = lo + item / d, j = item % d;
    const int e = plan.entry_expert[i];
    const T* wd = pool + ((size_t)plan.entry_slot[i] * L + layer) * blob_elems + gu2 + (size_t)j * d_ff;
    const int cnt = plan.exp_count[e];
    const int* pl = plan.pair_list + plan.exp_offset[e];
    for (int p0 = 0; p0 < cnt; p0 += 4) {
      const int np = min(4, cnt - p0);
      int pr[4];
      float acc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
      for (int q = 0; q < 4; ++q) pr[q] = q < np ? pl[p0 + q] : 0;
      for (int c = lane * N; c < d_ff; c += 32 * N) {
        float wv[N];
        Chunk<T>::load_stream(wd + c, wv);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          if (q < np) {
            const float* ap = act + (size_t)pr[q] * d_ff + c;
#pragma unroll
            for (int j4 = 0; j4 < N; j4 += 4) {
              const float4 av = *reinterpret_cast<const float4*>(ap + j4);
              acc[q] = fmaf(wv[j4], av.x, acc[q]); acc[q] = fmaf(wv[j4 + 1], av.y, acc[q]);
              acc[q] = fmaf(wv[j4 + 2], av.z, acc[q]); acc[q] = fmaf(wv[j4 + 3], av.w, acc[q]);
            }
          }
        }
      }
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const float y = warp_sum(acc[q]);
        if (q < np && lane == 0) ystage[(size_t)pr[q] * d + j] = y;
      }
    }
  }
}

// out[t, j] = sum_i w[t,i] * ystage[t*k+i, j] in rank order (fp32), stored in the model dtype.
// If x_res != nullptr also writes x_next = x_res + out with the rounding of DESIGN.md O3.
template <typename T>
__global__ void __launch_bounds__(256) combine_kernel(const float* __restrict__ ystage, const float* __restrict__ w,
                                                      T* __restrict__ out, const T* __restrict__ x_res,
                                                      T* __restrict__ x_next, int n_tokens, int d, int k) {
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (size_t)n_tokens * d) return;
  const int t = (int)(idx / d), j = (int)(idx % d);
  float acc = 0.f;
  for (int i = 0; i < k; ++i) acc = fmaf(w[(size_t)t * k + i], ystage[((size_t)t * k + i) * d + j], acc);
  const T o = from_f32<T>(acc);
  out[idx] = o;
  if (x_res) x_next[idx] = from_f32<T>(to_f32<T>(x_res[idx]) + to_f32<T>(o));
}

template <typename T>
__global__ void __launch_bounds__(256) residual_add_kernel(const T* __restrict__ x, const T* __restrict__ y,
                                                           T* __restrict__ out, size_t n) {
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx < n) out[idx] = from_f32<T>(to_f32<T>(x[idx]) + to_f32<T>(y[idx]));
}

}  // namespace wisp
