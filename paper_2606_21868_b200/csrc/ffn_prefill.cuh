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

// fp8 experts (f4): in-slot layout of the codes and scales (decode_ffn.cuh) read element by element and dequantised on the way
// into shared memory, w = e4m3(code) * S[block] in fp32 -- the first correct prefill version of the quantised path.
__device__ __forceinline__ float e4m3_to_f32(unsigned char c) {
  return __half2float(__ushort_as_half((unsigned short)(cvt_e4m3x2_f16x2((uint16_t)c) & 0xffffu)));
}
__host__ __device__ __forceinline__ size_t tiled_down_index_f8(int j, int i, int d) {   // 8 outputs x 8 act columns per 64-byte core
  return ((size_t)(i >> 3) * (d >> 3) + (j >> 3)) * 64 + (size_t)(j & 7) * 8 + (i & 7);
}

// grid: x = row tiles (n_rows/64), y = pair tiles (ceil(max_pairs_per_expert/64)), z = wave entry slot (C)
// MODE 0: gate/up + SwiGLU (A rows gathered from x by token); MODE 1: down (A rows = act[pair]).
// F8: T is the hidden-state type (bf16), the weights are fp8 blobs of `blob_elems` BYTES with scales at s13_off / s2_off.
template <typename T, int MODE, bool F8 = false>
__global__ void __launch_bounds__(256) prefill_ffn_kernel(PlanPtrs plan, int wave, int C, const T* __restrict__ pool,
                                                          size_t blob_elems, int L, int layer,
                                                          const T* __restrict__ x, T* __restrict__ act,
                                                          float* __restrict__ ystage, int d, int d_ff, int k,
                                                          size_t s13_off = 0, size_t s2_off = 0) {
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
  // weights are read through the tiled in-slot layout (common.cuh): gate / up rows r0.., or down rows (outputs j) r0..
  constexpr int kc = F8 ? 16 : 16 / (int)sizeof(T);
  const unsigned char* blob8 = reinterpret_cast<const unsigned char*>(pool) + ((size_t)plan.entry_slot[i] * L + layer) * blob_elems * (F8 ? 1 : sizeof(T));
  const T* blob = reinterpret_cast<const T*>(blob8);
  const T* wg = blob;
  const T* wu = blob + (size_t)d_ff * d;
  const T* wd = blob + 2 * (size_t)d_ff * d;
  const float* s13 = reinterpret_cast<const float*>(blob8 + s13_off);   // [2 d_ff / 128][d / 128]
  const float* s2t = reinterpret_cast<const float*>(blob8 + s2_off);    // [d_ff / 128][d / 128]

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
      if constexpr (F8) {
        if (MODE == 0) {
          const size_t wi = tiled_gu_index(r0 + row, k0 + kk, d, kc);
          const int kb = (k0 + kk) >> 7;
          sW0[kk][row] = e4m3_to_f32(blob8[wi]) * s13[(size_t)((r0 + row) >> 7) * (d >> 7) + kb];
          sW1[kk][row] = e4m3_to_f32(blob8[(size_t)d_ff * d + wi]) * s13[(size_t)((d_ff + r0 + row) >> 7) * (d >> 7) + kb];
        } else {
          sW0[kk][row] = e4m3_to_f32(blob8[2 * (size_t)d_ff * d + tiled_down_index_f8(r0 + row, k0 + kk, d)]) *
                         s2t[(size_t)((k0 + kk) >> 7) * (d >> 7) + ((r0 + row) >> 7)];
        }
      } else if (MODE == 0) {
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
  // four consecutive columns per thread (d % 4 == 0): the k float4 loads of a thread are independent and in flight together;
  // per element the arithmetic is the scalar chain (fmaf in rank order from 0.f)
  const size_t idx4 = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx4 * 4 >= (size_t)n_tokens * d) return;
  const int t = (int)(idx4 * 4 / d), j = (int)(idx4 * 4 % d);
  float acc[4] = {0.f, 0.f, 0.f, 0.f};
  const float4* src = reinterpret_cast<const float4*>(ystage + (size_t)t * k * d + j);
  for (int i0 = 0; i0 < k; i0 += 8) {
    float4 v[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) v[u] = __ldcs(src + (size_t)min(i0 + u, k - 1) * (d / 4));
#pragma unroll
    for (int u = 0; u < 8; ++u)
      if (i0 + u < k) {
        const float wi = w[(size_t)t * k + i0 + u];
        acc[0] = fmaf(wi, v[u].x, acc[0]); acc[1] = fmaf(wi, v[u].y, acc[1]);
        acc[2] = fmaf(wi, v[u].z, acc[2]); acc[3] = fmaf(wi, v[u].w, acc[3]);
      }
  }
  const size_t idx = idx4 * 4;
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    const T o = from_f32<T>(acc[c]);
    out[idx + c] = o;
    if (x_res) x_next[idx + c] = from_f32<T>(to_f32<T>(x_res[idx + c]) + to_f32<T>(o));
  }
}

}  // namespace wisp
