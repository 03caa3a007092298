// decode_combine.cuh -- the reduce-scatter half of a decode layer: ordered combine (+ residual) of the FFN chunk partials
// and the NEXT layer's router logits, both distributed over the grid in 16-column slices of the hidden state.
//
//   y_{t,i}[j]  = sum_{c = 0..NC-1} P[pos(t,i)][c][j]      8 groups of NC/8 consecutive chunks: inside a group ascending c
//                                                           (fp32 add chain from the first partial), then the 8 group sums
//                                                           ascending
//   out_t[j]    = sum_{i = 0..k-1} w[t,i] * y_{t,i}[j]      fmaf in rank order from 0.f, stored in the model dtype (a4, G21)
//   x'_t[j]     = x_t[j] + out_t[j]                         fp32 add of the two model-dtype values, stored in the model dtype (O3)
//   z_e        += sum_{j in slice} W_r[e][j] * x'_t[j]      fmaf in ascending j from 0.f per slice, then added to the logit
//                                                           accumulator as a 2^-32 fixed-point integer (a1)
// The logit accumulator is an int64 per (token, expert): integer addition is associative, so the all-reduce of the
// 16-column partial logits over the grid is bit-reproducible whatever order the CTAs' `red.add.u64` arrive in, and it needs
// no second grid-wide exchange: after one barrier every CTA reads E words per token.  (A logit partial is O(1); 2^-32
// resolution is five orders of magnitude below fp32 rounding of the logit itself.)
#pragma once
#include "common.cuh"

namespace wisp {

constexpr int kSliceCols = 16;
// The accumulator of a (token, expert) exists in kZfixCopies copies; a CTA adds into copy blockIdx.x % kZfixCopies and the reader
// sums the copies (integers: still one value whatever the order).  ~128 CTAs adding to the SAME word serialise in L2 at ~27 clk per
// add (B300_MICROARCH.md: cyc/op = n_conc * 32 * 0.854); four copies cut that queue to a quarter.
constexpr int kZfixCopies = 4;
__host__ __device__ __forceinline__ size_t zfix_plane(int E) { return (size_t)kDecodeMaxTokens * E; }   // words per (parity, copy)
// An accumulator word = (sum of the 2^-32 fixed-point partial logits) << 10 | number of partials added so far (< 1024 per copy:
// d / 16 / kZfixCopies).  The count makes the word self-describing: a reader that knows how many partials a copy receives can tell
// from the word alone that its sum is complete -- the fused kernel polls the words instead of crossing a grid barrier (E) and
// then reading them.
constexpr float kLogitFixScale = 4294967296.f;           // 2^32
constexpr float kLogitFixInv = 1.0f / 4294967296.f;       // 2^-32 (exact)
__device__ __forceinline__ long long logit_to_fix(float v) {
  const float s = v * kLogitFixScale;
  if (!(fabsf(s) < 2.2e15f)) return s > 0.f ? (1ll << 51) : -(1ll << 51);   // |v| >= 2^19 or non-finite (G23): saturate, stay defined
  return __float2ll_rn(s);
}
constexpr int kZfixCountBits = 10;
__device__ __forceinline__ unsigned long long zfix_pack(float v) { return ((unsigned long long)logit_to_fix(v) << kZfixCountBits) + 1ull; }   // one partial
__device__ __forceinline__ unsigned long long zfix_pack_uncounted(float v) { return (unsigned long long)logit_to_fix(v) << kZfixCountBits; }
__device__ __forceinline__ long long zfix_value(long long word) { return word >> kZfixCountBits; }
__device__ __forceinline__ int zfix_count(long long word) { return (int)(word & ((1 << kZfixCountBits) - 1)); }
__device__ __forceinline__ long long zfix_sum(const long long* z0, size_t plane) {       // z0 = the word in copy 0; complete words
  long long v = 0;
#pragma unroll
  for (int c = 0; c < kZfixCopies; ++c) v += zfix_value(__ldcg(z0 + c * plane));
  return v;
}
// one rounding (int64 -> fp32), an exact scaling, one fp32 add; no fp64 on the routing chain
__device__ __forceinline__ float logit_from_fix(long long f, float bias) { return __ll2float_rn(f) * kLogitFixInv + bias; }

// Partial logits of one 16-column slice of token t's hidden state (xn[16], fp32 images of the model-dtype values) for all
// experts, added into zfix[t][e].  w16: rows j0 .. j0+15 of this layer's router weights TRANSPOSED ([d][E], model dtype), in
// global memory or staged in shared memory.
template <typename T>
__device__ __forceinline__ void slice_logits(const T* w16, const float* xn, int E, long long* zfix_t, int tid, int nthr) {
  for (int e = tid; e < E; e += nthr) {
    float zp = 0.f;
#pragma unroll
    for (int jj = 0; jj < kSliceCols; ++jj) zp = fmaf(to_f32<T>(w16[(size_t)jj * E + e]), xn[jj], zp);
    atomicAdd(reinterpret_cast<unsigned long long*>(zfix_t + e), zfix_pack(zp));
  }
}

// The same for `ns` tokens at once (their fp32 images in xn[s][16]): each thread reads its 16 weights once.  Per token the
// arithmetic is slice_logits' (fmaf in ascending j from 0.f).
template <typename T, int S>
__device__ __forceinline__ void slice_logits_multi(const T* w16, const float* xn, int ns, int E, long long* zfix_t0, int tid, int nthr) {
  for (int e = tid; e < E; e += nthr) {
    float wv[kSliceCols];
#pragma unroll
    for (int jj = 0; jj < kSliceCols; ++jj) wv[jj] = to_f32<T>(w16[(size_t)jj * E + e]);
#pragma unroll
    for (int s = 0; s < S; ++s) {
      if (s < ns) {
        float zp = 0.f;
#pragma unroll
        for (int jj = 0; jj < kSliceCols; ++jj) zp = fmaf(wv[jj], xn[s * kSliceCols + jj], zp);
        atomicAdd(reinterpret_cast<unsigned long long*>(zfix_t0 + (size_t)s * E + e), zfix_pack(zp));
      }
    }
  }
}

struct CombineArgs {
  const float* partial;      // P [pair position][NC][d]
  int n_chunks, d, k;
  const float* topw;         // [T][k] routing weights (rank order)
  const int* pair_pos;       // [T][k] position of pair (t, rank) in the expert-sorted order
};

// One slice (token t, columns j0 .. j0+15) by 256 threads synchronising on named barrier `bar`.
//   x_row  : token t's current hidden state (model dtype) or nullptr (no residual: the result is out_t itself)
//   dst_row: where the result row goes (global, model dtype)
//   s_yg   : 8 * 8 * 16 floats, s_y: kMaxTopK * 16 floats, s_xn: 16 floats (receives the fp32 image of the stored result)
template <typename T, int U = 16>
__device__ __forceinline__ void combine_slice(const CombineArgs& a, int t, int j0, const T* x_row, T* dst_row, float* s_yg, float* s_y,
                                              float* s_xn, int bar) {
  const int tid = threadIdx.x, grp = tid >> 5, lane = tid & 31, ri = lane >> 2, j4 = (lane & 3) * 4;
  const int per = a.n_chunks >> 3;
  for (int i0 = 0; i0 < a.k; i0 += 8) {
    const int rank = i0 + ri;
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    if (rank < a.k) {
      const int pos = a.pair_pos[t * a.k + rank];
      const float* src = a.partial + ((size_t)pos * a.n_chunks + (size_t)grp * per) * a.d + j0 + j4;
      for (int c0 = 0; c0 < per; c0 += U) {                  // up to U independent L2 reads in flight, added in ascending c
        float4 v[U];
#pragma unroll
        for (int u = 0; u < U; ++u)                            // unpredicated (index clamped) so that all loads issue before the first add
          v[u] = __ldcg(reinterpret_cast<const float4*>(src + (size_t)min(c0 + u, per - 1) * a.d));
#pragma unroll
        for (int u = 0; u < U; ++u)
          if (c0 + u < per) {
            if (c0 + u == 0) acc = v[0];
            else { acc.x += v[u].x; acc.y += v[u].y; acc.z += v[u].z; acc.w += v[u].w; }
          }
      }
    }
    *reinterpret_cast<float4*>(s_yg + (grp * 8 + ri) * kSliceCols + j4) = acc;
    asm volatile("bar.sync %0, 256;" ::"r"(bar) : "memory");
    if (tid < 32 && rank < a.k) {
      float4 y = *reinterpret_cast<const float4*>(s_yg + ri * kSliceCols + j4);
#pragma unroll
      for (int g = 1; g < 8; ++g) {
        const float4 v = *reinterpret_cast<const float4*>(s_yg + (g * 8 + ri) * kSliceCols + j4);
        y.x += v.x; y.y += v.y; y.z += v.z; y.w += v.w;
      }
      *reinterpret_cast<float4*>(s_y + rank * kSliceCols + j4) = y;
    }
    asm volatile("bar.sync %0, 256;" ::"r"(bar) : "memory");
  }
  if (tid < kSliceCols) {
    float acc = 0.f;
    for (int i = 0; i < a.k; ++i) acc = fmaf(a.topw[t * a.k + i], s_y[i * kSliceCols + tid], acc);
    T o = from_f32<T>(acc);
    if (x_row) o = from_f32<T>(to_f32<T>(x_row[j0 + tid]) + to_f32<T>(o));
    dst_row[j0 + tid] = o;
    s_xn[tid] = to_f32<T>(o);
  }
  asm volatile("bar.sync %0, 256;" ::"r"(bar) : "memory");
}

// The slices (t0 .. t0+ns-1, columns j0 .. j0+15) of up to S tokens in ONE pass: the partial loads of all of them are in flight
// together (a decode batch's combine is bound by L2 round trips, not by bytes).  Per slice the arithmetic, and so every bit, is
// combine_slice's: 8 groups of consecutive chunks (warp = group), ascending inside a group from its first partial, groups
// ascending, ranks in order.  U: chunk loads per thread and slice in flight.
//   x_base / xs_pitch: the tokens' hidden states (row t at x_base + t * xs_pitch) or nullptr; dst_base: result rows [t][d]
//   s_yg: S * 8 * 8 * 16 floats, s_y: S * kMaxTopK * 16 floats, s_xn: S * 16 floats
template <typename T, int S, int U>
__device__ __forceinline__ void combine_tokens(const CombineArgs& a, int t0, int ns, int j0, const T* x_base, int xs_pitch, T* dst_base,
                                               float* s_yg, float* s_y, float* s_xn, int bar) {
  const int tid = threadIdx.x, grp = tid >> 5, lane = tid & 31, ri = lane >> 2, j4 = (lane & 3) * 4;
  const int per = a.n_chunks >> 3;
  for (int i0 = 0; i0 < a.k; i0 += 8) {
    const int rank = i0 + ri;
    float4 acc[S];
#pragma unroll
    for (int s = 0; s < S; ++s) acc[s] = make_float4(0.f, 0.f, 0.f, 0.f);
    if (rank < a.k) {
      const float* src[S];
#pragma unroll
      for (int s = 0; s < S; ++s) {
        const int pos = a.pair_pos[min(t0 + s, t0 + ns - 1) * a.k + rank];
        src[s] = a.partial + ((size_t)pos * a.n_chunks + (size_t)grp * per) * a.d + j0 + j4;
      }
      for (int c0 = 0; c0 < per; c0 += U) {
        float4 v[S][U];
#pragma unroll
        for (int s = 0; s < S; ++s)
#pragma unroll
          for (int u = 0; u < U; ++u) v[s][u] = __ldcg(reinterpret_cast<const float4*>(src[s] + (size_t)min(c0 + u, per - 1) * a.d));
#pragma unroll
        for (int s = 0; s < S; ++s)
#pragma unroll
          for (int u = 0; u < U; ++u)
            if (c0 + u < per) {
              if (c0 + u == 0) acc[s] = v[s][0];
              else { acc[s].x += v[s][u].x; acc[s].y += v[s][u].y; acc[s].z += v[s][u].z; acc[s].w += v[s][u].w; }
            }
      }
    }
#pragma unroll
    for (int s = 0; s < S; ++s) *reinterpret_cast<float4*>(s_yg + ((s * 8 + grp) * 8 + ri) * kSliceCols + j4) = acc[s];
    asm volatile("bar.sync %0, 256;" ::"r"(bar) : "memory");
    if (tid < 32 * ns && rank < a.k) {                          // warp s adds the 8 group sums of slice s, ascending
      const float* yg = s_yg + (size_t)grp * 8 * 8 * kSliceCols;
      float4 y = *reinterpret_cast<const float4*>(yg + ri * kSliceCols + j4);
#pragma unroll
      for (int g = 1; g < 8; ++g) {
        const float4 v = *reinterpret_cast<const float4*>(yg + (g * 8 + ri) * kSliceCols + j4);
        y.x += v.x; y.y += v.y; y.z += v.z; y.w += v.w;
      }
      *reinterpret_cast<float4*>(s_y + ((size_t)grp * kMaxTopK + rank) * kSliceCols + j4) = y;
    }
    asm volatile("bar.sync %0, 256;" ::"r"(bar) : "memory");
  }
  if (tid < kSliceCols * ns) {
    const int s = tid >> 4, col = tid & 15, t = t0 + s;
    float acc = 0.f;
    for (int i = 0; i < a.k; ++i) acc = fmaf(a.topw[t * a.k + i], s_y[((size_t)s * kMaxTopK + i) * kSliceCols + col], acc);
    T o = from_f32<T>(acc);
    if (x_base) o = from_f32<T>(to_f32<T>(x_base[(size_t)t * xs_pitch + j0 + col]) + to_f32<T>(o));
    dst_base[(size_t)t * a.d + j0 + col] = o;
    s_xn[s * kSliceCols + col] = to_f32<T>(o);
  }
  asm volatile("bar.sync %0, 256;" ::"r"(bar) : "memory");
}

}  // namespace wisp
