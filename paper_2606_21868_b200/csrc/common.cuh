// common.cuh -- shared device helpers and plain structs of libwisp (sm_100a only).
//
// Canonical dot-product order: every (weight row, token) dot product in the
// router and the decode FFN is computed by ONE warp: lane l accumulates the 16-byte chunks l, l+32,
// l+64, ... of the row in that order, elements of a chunk in ascending order, with fmaf into a single
// fp32 accumulator, and the 32 lane sums are combined by an xor-butterfly (16, 8, 4, 2, 1).  The order
// does not depend on the slot, the wave, the number of tokens in the call or the launch geometry, which
// is what makes outputs byte-identical across budgets (parity (b)).
#pragma once
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/wisp.h"
#include "ptx.cuh"

namespace wisp {

typedef unsigned long long u64;

constexpr int kMaxExperts = 1024;
constexpr int kMaxTopK = 32;
constexpr int kDecodeMaxTokens = 8;   // n_tokens <= this -> GEMV path; above -> grouped GEMM path

// ---- 16-byte chunk loads widened to fp32 ------------------------------------------------------------
template <typename T> struct Chunk;
template <> struct Chunk<float> {
  static constexpr int N = 4;
  __device__ __forceinline__ static void load(const float* p, float (&v)[4]) {
    float4 r = *reinterpret_cast<const float4*>(p);
    v[0] = r.x; v[1] = r.y; v[2] = r.z; v[3] = r.w;
  }
  __device__ __forceinline__ static void load_stream(const float* p, float (&v)[4]) {
    float4 r = __ldcs(reinterpret_cast<const float4*>(p));
    v[0] = r.x; v[1] = r.y; v[2] = r.z; v[3] = r.w;
  }
};
__device__ __forceinline__ void widen_bf16x8(const uint4& r, float (&v)[8]) {
  v[0] = __uint_as_float(r.x << 16); v[1] = __uint_as_float(r.x & 0xffff0000u);
  v[2] = __uint_as_float(r.y << 16); v[3] = __uint_as_float(r.y & 0xffff0000u);
  v[4] = __uint_as_float(r.z << 16); v[5] = __uint_as_float(r.z & 0xffff0000u);
  v[6] = __uint_as_float(r.w << 16); v[7] = __uint_as_float(r.w & 0xffff0000u);
}
template <> struct Chunk<__nv_bfloat16> {
  static constexpr int N = 8;
  __device__ __forceinline__ static void load(const __nv_bfloat16* p, float (&v)[8]) {
    widen_bf16x8(*reinterpret_cast<const uint4*>(p), v);
  }
  __device__ __forceinline__ static void load_stream(const __nv_bfloat16* p, float (&v)[8]) {
    widen_bf16x8(__ldcs(reinterpret_cast<const uint4*>(p)), v);
  }
};

template <typename T> struct ChunkW;   // a 16-byte weight chunk widened to fp32
template <> struct ChunkW<float> {
  static constexpr int N = 4;
  __device__ __forceinline__ static void widen(const uint4& r, float (&v)[4]) {
    v[0] = __uint_as_float(r.x); v[1] = __uint_as_float(r.y); v[2] = __uint_as_float(r.z); v[3] = __uint_as_float(r.w);
  }
};
template <> struct ChunkW<__nv_bfloat16> {
  static constexpr int N = 8;
  __device__ __forceinline__ static void widen(const uint4& r, float (&v)[8]) { widen_bf16x8(r, v); }
};

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

template <typename T> __device__ __forceinline__ float to_f32(T v);
template <> __device__ __forceinline__ float to_f32<float>(float v) { return v; }
template <> __device__ __forceinline__ float to_f32<__nv_bfloat16>(__nv_bfloat16 v) { return __bfloat162float(v); }
template <typename T> __device__ __forceinline__ T from_f32(float v);
template <> __device__ __forceinline__ float from_f32<float>(float v) { return v; }
template <> __device__ __forceinline__ __nv_bfloat16 from_f32<__nv_bfloat16>(float v) { return __float2bfloat16_rn(v); }

__device__ __forceinline__ float silu_f(float v) { return v / (1.0f + expf(-v)); }

// ---- in-slot weight layout ("core-matrix tiled") ------------------------------------------
// The library re-tiles the caller's canonical blob [gate | up | down] (row-major out x in) once, at registration, into
// 8-row x 16-byte core matrices (128 contiguous bytes each; kc = 16 / sizeof(dtype) elements per row of a core):
//   gate, up  [d_ff x d]   : core (r/8, k/kc)  at ((r/8) * (d/kc)  + k/kc) * 128 B   -> 8 act rows x all of d are contiguous
//   down      [d x d_ff]   : core (j/8, i/kc)  at ((i/kc) * (d/8)  + j/8 ) * 128 B   -> 8 act columns x all of d are contiguous
// inside a core: row (r%8 | j%8) at 16 B * row, element (k%kc | i%kc).  One decode work unit (8 act rows: their gate rows, up
// rows and down columns) is then three contiguous pieces that 1-D TMA bulk copies fetch whole, ldmatrix reads without bank
// conflicts, and the prefill tcgen05 kernel consumes as the canonical no-swizzle K-major operand layout.  Master bytes == slot
// bytes: the same tiling lives in the pinned master and in every slot.
__host__ __device__ __forceinline__ size_t tiled_gu_index(int r, int k, int d, int kc) {
  return ((size_t)(r >> 3) * (d / kc) + k / kc) * (8 * kc) + (size_t)(r & 7) * kc + k % kc;
}
__host__ __device__ __forceinline__ size_t tiled_down_index(int j, int i, int d, int kc) {
  return ((size_t)(i / kc) * (d >> 3) + (j >> 3)) * (8 * kc) + (size_t)(j & 7) * kc + i % kc;
}

// ---- the per-forward plan written by the residency kernel ------------------------------------------
// hdr[0] = n_waves, hdr[1] = n_ref (|R|), hdr[2] = n_miss, hdr[3] = n_pairs.  Entries are in wave order
// (ascending expert id; wave w = entries [w*C, min(n_ref, (w+1)*C)) ).
struct PlanPtrs {
  int* hdr;
  int* entry_expert;   // [E]
  int* entry_slot;     // [E]
  int* entry_miss;     // [E]  1 = fetched in this step
  int* exp_count;      // [E]  (token, rank) pairs routed to expert e
  int* exp_offset;     // [E+1] exclusive prefix of exp_count over ascending e
  int* pair_list;      // [n_pairs] pair indices (t*k + rank) grouped by expert, ascending inside a group
  // decode path only (nullable): the order in which the FFN takes the entries of a wave, and the inverse of pair_list
  int* unit_entry;     // [E]  per wave segment [w*C, ...): entry indices, this step's misses first (their host reads start at once)
  int* pair_pos;       // [n_pairs] pair_pos[pair_list[p]] = p: position of a (token, rank) pair in the expert-sorted order
};

// Host-visible copy of the plan for the MEMCPY miss path (mapped pinned memory).
struct HostPlan {
  int n_waves, n_ref, n_miss, n_pairs;
  int entry_expert[kMaxExperts];
  int entry_slot[kMaxExperts];
  int entry_miss[kMaxExperts];
};

// Per-layer residency state in device memory (pi, pi^-1, tau, clock of Algorithm 1; f for LFU).
struct LayerState {
  int* pi;        // [E] expert -> slot, -1 absent  (pi_dev)
  int* pi_inv;    // [E] slot -> expert, -1 empty   (first C entries live)
  u64* tau;       // [E] per-slot tick
  u64* freq;      // [E] per-expert LFU count
  u64* scal;      // [8] 0 clock, 1 step, 2 hits, 3 misses, 4 evictions, 5 references
  u64* last_pos;  // [E] MV-WSA: linear position of the last reference (0 = never)
  u64* hist;      // [E+2] MV-WSA: reuse-distance counts since the last read; [E+1] = cold/inf
};

}  // namespace wisp
