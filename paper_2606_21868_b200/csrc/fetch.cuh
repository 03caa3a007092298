// fetch.cuh -- (a3) demand fetch, device-initiated variant: a copy kernel that reads the mapped pinned
// host master over the host link and writes the victim slots (Alg. 1 line 6).  The
// cudaMemcpyAsync variant lives in wisp.cu.  No arithmetic: slot bytes == master bytes.
#pragma once
#include "common.cuh"

namespace wisp {

constexpr int kFetchThreads = 256;
constexpr int kFetchUnroll = 8;                                   // 16-byte loads in flight per thread
constexpr size_t kFetchChunk = (size_t)kFetchThreads * kFetchUnroll * 16;   // 32 KiB per CTA iteration

// Copies every miss of wave `wave` of the current plan.  master = mapped host pointer of the layer's E
// blobs; pool = arena base; slot s of this layer is at pool + ((size_t)s * L + layer) * M_e.
__global__ void __launch_bounds__(kFetchThreads) fetch_zerocopy_kernel(PlanPtrs plan, int wave, int C,
                                                                       const uint4* __restrict__ master,
                                                                       uint4* __restrict__ pool, size_t blob_vec,
                                                                       int L, int layer) {
  if (wave >= plan.hdr[0] || plan.hdr[2] == 0) return;       // nothing missed in this step: no walk over the entries
  const int lo = wave * C, hi = min(plan.hdr[1], lo + C);
  const size_t chunk_vec = kFetchChunk / 16;
  const size_t chunks_per_blob = (blob_vec + chunk_vec - 1) / chunk_vec;
  size_t miss_no = 0;
  for (int i = lo; i < hi; ++i) {
    if (!plan.entry_miss[i]) continue;
    const uint4* src = master + (size_t)plan.entry_expert[i] * blob_vec;
    uint4* dst = pool + ((size_t)plan.entry_slot[i] * L + layer) * blob_vec;
    // CTAs take chunks round-robin across ALL misses of the wave so every miss uses the whole grid
    for (size_t c = (blockIdx.x + gridDim.x - (miss_no * chunks_per_blob) % gridDim.x) % gridDim.x;
         c < chunks_per_blob; c += gridDim.x) {
      const size_t base = c * chunk_vec + threadIdx.x;
      uint4 v[kFetchUnroll];
#pragma unroll
      for (int u = 0; u < kFetchUnroll; ++u) {
        const size_t idx = base + (size_t)u * kFetchThreads;
        if (idx < blob_vec) v[u] = __ldcs(src + idx);
      }
#pragma unroll
      for (int u = 0; u < kFetchUnroll; ++u) {
        const size_t idx = base + (size_t)u * kFetchThreads;
        if (idx < blob_vec) dst[idx] = v[u];
      }
    }
    ++miss_no;
  }
}

// Device-to-device slot moves of a resize (src, dst pairs), grid.y = move index.
__global__ void __launch_bounds__(256) move_slots_kernel(const int* __restrict__ moves, const int* __restrict__ n_moves,
                                                         uint4* __restrict__ pool, size_t blob_vec, int L, int layer) {
  const int m = blockIdx.y;
  if (m >= *n_moves) return;
  const uint4* src = pool + ((size_t)moves[2 * m] * L + layer) * blob_vec;
  uint4* dst = pool + ((size_t)moves[2 * m + 1] * L + layer) * blob_vec;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < blob_vec; i += (size_t)gridDim.x * blockDim.x)
    dst[i] = src[i];
}

// Exactness invariant: slot bytes == master bytes for every occupied slot.  grid.y = slot.
__global__ void __launch_bounds__(256) verify_pool_kernel(const int* __restrict__ pi_inv, const uint4* __restrict__ master,
                                                          const uint4* __restrict__ pool, size_t blob_vec, int L, int layer,
                                                          int* __restrict__ bad_slots) {
  const int s = blockIdx.y;
  const int e = pi_inv[s];
  if (e < 0) return;
  const uint4* a = master + (size_t)e * blob_vec;
  const uint4* b = pool + ((size_t)s * L + layer) * blob_vec;
  int bad = 0;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < blob_vec; i += (size_t)gridDim.x * blockDim.x) {
    const uint4 x = a[i], y = b[i];
    bad |= (x.x != y.x) | (x.y != y.y) | (x.z != y.z) | (x.w != y.w);
  }
  if (bad) atomicOr(&bad_slots[s], 1);
}

}  // namespace wisp
