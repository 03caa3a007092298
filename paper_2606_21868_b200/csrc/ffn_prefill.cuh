// ffn_prefill.cuh -- (a4/a5) grouped expert FFN for many tokens (prefill): per wave entry (expert in a
// slot) a GEMM over that expert's gathered token rows.  First correct version: shared-memory tiled fp32
// FMA GEMM with a fixed K order (deterministic, independent of wave / slot / tile position).
//   act[pair, r]  = silu(<G[r], x_t>) * <U[r], x_t>      stored in the model dtype
//   ystage[pair, j] = <D[j], act[pair]>                   fp32
#pragma once
#include "common.cuh"

namespace wisp {

constexpr int kPfTile = 64;    // 64 pairs x 64 weight rows per CTA
constexpr int kPfK = 32;

// grid: x = row tiles (n_rows/64), y = pair tiles (ceil(max_pairs_per_expert/64)), z = wave entry slot (C)
// MODE 0: gate/up + SwiGLU (A rows gathered from x by token); MODE 1: down (A rows = act[pair]).
template <typename T, int MODE>
__global__ void __launch_bounds__(256) prefill_ffn_kernel(PlanPtrs plan, int wave, int C, const T* __restrict__ pool,
                                                          size_t blob_elems, int L, int layer,
                                                          const T* __restrict__ x, T* __restrict__ act,
                                                          float* __restrict__ ystage, int d, int d_ff, int k) {
  if (wave >= plan.hdr[0]) return;
  const int lo = wave * C, nw = min(plan.hdr[1], lo + C) - lo;
  if ((int)blockIdx.z >= nw) return;
  const int i = lo + blockIdx.z;
  const int e = plan.entry_expert[i];
  const int cnt = plan.exp_count[e];
  const int p0 = blockIdx.y * kPfTile;
  if (p0 >= cnt) return;
  const int* pl = plan.pair_list + plan.exp_offset[e];
  const int K = MODE == 0 ? d : d_ff;
  const int r0 = blockIdx.x * kPfTile;
  const T* blob = pool + ((size_t)plan.entry_slot[i] * L + layer) * blob_elems;
  // weights are read through the tiled in-slot layout (common.cuh): gate / up rows r0.., or down rows (outputs j) r0..
  constexpr int kc = 16 / (int)sizeof(T);
  const T* wg = blob;
  const T* wu = blob + (size_t)d_ff * d;
  const T* wd = blob + 2 * (size_t)d_ff * d;

  __shared__ float sA[kPfK][kPfTile + 1];
  __shared__ float sW0[kPfK][kPfTile + 1];
  __shared__ float sW1[MODE == 0 ? kPfK : 1][kPfTile + 1];
  __shared__ int s_pair[kPfTile];
  const int tid = threadIdx.x;
  if (tid < kPfTile) s_pair[tid] = (p0 + tid < cnt) ? pl[p0 + tid] : -1;
  __syncthreads();
  const int tx = tid & 15, ty = tid >> 4;     // 16 x 16 threads, each 4 pairs x 4 rows
  float c0[4][4] = {}, c1[4][4] = {};
  for (int k0 = 0; k0 < K; k0 += kPfK) {
    // load tiles: 64 x 32 elements each, 256 threads -> 8 elements per thread
    for (int idx = tid; idx < kPfTile * kPfK; idx += 256) {
      const int row = idx / kPfK, kk = idx % kPfK;
      const int pr = s_pair[row];
      float av = 0.f;
      if (pr >= 0) av = MODE == 0 ? to_f32<T>(x[(size_t)(pr / k) * d + k0 + kk]) : to_f32<T>(act[(size_t)pr * d_ff + k0 + kk]);
      sA[kk][row] = av;
      if (MODE == 0) {
        const size_t wi = tiled_gu_index(r0 + row, k0 + kk, d, kc);
        sW0[kk][row] = to_f32<T>(wg[wi]);
        sW1[kk][row] = to_f32<T>(wu[wi]);
      } else {
        sW0[kk][row] = to_f32<T>(wd[tiled_down_index(r0 + row, k0 + kk, d, kc)]);
      }
    }
    __syncthreads();
#pragma unroll 8
    for (int kk = 0; kk < kPfK; ++kk) {
      float a[4], b0[4], b1[4];
#pragma unroll
      for (int q = 0; q < 4; ++q) { a[q] = sA[kk][ty * 4 + q]; b0[q] = sW0[kk][tx * 4 + q]; if (MODE == 0) b1[q] = sW1[kk][tx * 4 + q]; }
#pragma unroll
      for (int p = 0; p < 4; ++p)
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          c0[p][q] = fmaf(a[p], b0[q], c0[p][q]);
          if (MODE == 0) c1[p][q] = fmaf(a[p], b1[q], c1[p][q]);
        }
    }
    __syncthreads();
  }
#pragma unroll
  for (int p = 0; p < 4; ++p) {
    const int pr = s_pair[ty * 4 + p];
    if (pr < 0) continue;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const int r = r0 + tx * 4 + q;
      if (MODE == 0) act[(size_t)pr * d_ff + r] = from_f32<T>(silu_f(c0[p][q]) * c1[p][q]);
      else ystage[(size_t)pr * d + r] = c0[p][q];
    }
  }
}

// out[t, j] = sum_i w[t,i] * ystage[t*k+i, j] in rank order (fmaf from 0.f, fp32), stored in the model dtype; the optional
// residual successor x_next = x + out uses the rounding of DESIGN.md O3.  Prefill / overflow staging path (a5): the grouped
// GEMMs leave y per (token, rank) pair in ystage [T*k][d].
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

}  // namespace wisp
