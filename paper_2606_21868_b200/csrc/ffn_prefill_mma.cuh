// ffn_prefill_mma.cuh -- (a4, prefill) grouped expert FFN over slot-indexed experts on the 5th-generation tensor
// cores (tcgen05.mma, accumulators in TMEM, operands staged by TMA with the 128-byte swizzle).  bf16 only; the fp32
// model dtype keeps the plain tiled kernel of ffn_prefill.cuh.  The paper runs the engine's unmodified fused-MoE
// kernel here; this is the part of the path that really is a dense contraction.
//
// Per wave entry (expert e resident in slot s, n_e routed (token, rank) pairs, sorted positions pos0..pos0+n_e-1):
//   GEMM 1 (MODE 0):  Hg = G_s Xe^T, Hu = U_s Xe^T     [128 weight rows x NT tokens] per CTA, K = d_model
//                     act[pos, r] = silu(Hg[r, pos]) * Hu[r, pos]   (bf16, sorted-pair order, G21)
//   GEMM 2 (MODE 1):  Y = D_s act_e^T                   [128 rows x NT tokens], K = d_ff  -> ystage[pair, r] fp32
// "Swap AB": the weight rows are the MMA M dimension (always 128 full rows), the ragged token count is N.
// Operands are K-major.  A tiles come straight from the slot: the in-slot layout (common.cuh) stores every matrix as
// 8-row x 16-byte core matrices of 128 contiguous bytes, which is the canonical NO-SWIZZLE K-major UMMA operand layout, so a
// 4-D tensor map (64 elements of a core, core column, core row, blob index = slot*L + layer) drops a 128 x 64 tile into shared
// memory ready for the descriptor (gate/up: cores of a row group adjacent along K; down: cores of an act-column block
// adjacent along M).  B tiles come from the gathered token rows xg / the act buffer with the 128-byte swizzle.
// Warp roles (192 threads): warp 0 = TMA producer, warp 1 = TMEM allocator + MMA issuer, warps 2..5 = epilogue.
// Determinism (parity (b)): a column (token) of the accumulator depends only on that token's row and the weight
// tile, the K order is fixed, and nothing depends on the slot, the wave or the other tokens of the tile.
#pragma once
#include <cuda.h>

#include "common.cuh"

namespace wisp {

constexpr int kMmaThreads = 192;
constexpr int kMmaM = 128;        // weight rows per CTA tile (UMMA_M)
constexpr int kMmaNT = 128;       // tokens per CTA tile (UMMA_N <= 128)
constexpr int kMmaBK = 64;        // K elements per stage = one 128-byte swizzle atom of bf16
constexpr int kMmaTileBytes = kMmaM * kMmaBK * 2;   // 16 KiB: [128 rows][128 B]

struct MmaArgs {
  PlanPtrs plan;
  int wave, C, L, layer;
  int d, dff, k;
  __nv_bfloat16* act;     // [n_pairs][dff] bf16, SORTED pair order (position = exp_offset[e] + j)
  float* ystage;          // [n_pairs][d] fp32, indexed by pair id (t*k + rank)
  // MODE 2 (router logits, a1 for prefill): z[t][e] = bias[e] + <W_r[e], x_t>, E a multiple of 128
  float* z;               // [n_tokens][E] fp32
  const float* bias;      // [E] of this layer
  int n_tokens, E;
  int b_rows;             // MODE 2: tokens per tile = rows of the B box (32: the router GEMM has few tiles, small ones fill the grid)
};

struct MmaTile { int pos0, nt, blob, r0; };
// tile t -> (first B row, valid B rows, weight blob, first weight row).  The work list holds one resolved item per
// (wave entry, token tile): int4 (first sorted pair position, valid pairs, slot of the expert, plan entry) -- ONE 16-byte load per
// tile (the chain work -> entry_expert -> exp_offset / exp_count / entry_slot cost each role ~2 us of dependent L2 loads per tile).
template <int MODE>
__device__ __forceinline__ MmaTile mma_tile(const MmaArgs& a, const int* work, int t, int RT) {
  MmaTile m;
  const int w = t / RT;
  m.r0 = (t % RT) * (MODE == 1 ? 2 * kMmaM : kMmaM);           // MODE 1: a tile is TWO 128-row blocks of the down matrix
  if (MODE == 2) {
    m.pos0 = w * a.b_rows; m.nt = min(a.b_rows, a.n_tokens - m.pos0); m.blob = a.layer;
  } else {
    const int4 it = __ldg(reinterpret_cast<const int4*>(work) + w);
    m.pos0 = it.x; m.nt = it.y; m.blob = it.z * a.L + a.layer;
  }
  return m;
}

// ---- PTX wrappers -----------------------------------------------------------------------------------------------
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* tm, int c0, int c1, uint32_t bar) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
               ::"r"(dst), "l"(tm), "r"(bar), "r"(c0), "r"(c1) : "memory");
}
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* tm, int c0, int c1, int c2, uint32_t bar) {
  asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
               ::"r"(dst), "l"(tm), "r"(bar), "r"(c0), "r"(c1), "r"(c2) : "memory");
}
__device__ __forceinline__ void tma_load_4d(uint32_t dst, const CUtensorMap* tm, int c0, int c1, int c2, int c3, uint32_t bar) {
  asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
               ::"r"(dst), "l"(tm), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}
__device__ __forceinline__ void tmem_alloc(uint32_t smem_dst, uint32_t cols) {
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_dst), "r"(cols) : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t cols) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(cols) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
// D[tmem] (+)= A[smem desc] * B[smem desc]^T, bf16 inputs, fp32 accumulate, issued by one thread
__device__ __forceinline__ void umma_bf16(uint32_t tmem_d, uint64_t desc_a, uint64_t desc_b, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\n"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n}"
      ::"r"(tmem_d), "l"(desc_a), "l"(desc_b), "r"(idesc), "r"(accumulate) : "memory");
}
// mbarrier arrive once every tcgen05.mma issued so far by this thread has completed
__device__ __forceinline__ void umma_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
// 16 consecutive fp32 columns of this thread's TMEM lane
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, float (&v)[16]) {
  uint32_t r[16];
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
                 "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
               : "r"(taddr) : "memory");
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
  for (int i = 0; i < 16; ++i) v[i] = __uint_as_float(r[i]);
}

// Shared-memory matrix descriptor of a K-major tile [rows][64 bf16] written by TMA with the 128-byte swizzle:
// 8-row groups are 1024 B apart (SBO), descriptor version 1 (sm_100), layout type 2 = SWIZZLE_128B.
__device__ __forceinline__ uint64_t umma_desc_sw128(uint32_t smem_addr) {
  uint64_t desc = 0;
  desc |= (uint64_t)((smem_addr >> 4) & 0x3fffu);            // start address, 16-byte units
  desc |= (uint64_t)1 << 16;                                 // leading byte offset (unused for swizzled K-major)
  desc |= (uint64_t)(1024u >> 4) << 32;                      // stride byte offset
  desc |= (uint64_t)1 << 46;                                 // version
  desc |= (uint64_t)2 << 61;                                 // SWIZZLE_128B
  return desc;
}
// Shared-memory matrix descriptor of a K-major tile stored as plain (unswizzled) core matrices of 8 rows x 16 bytes, 128
// contiguous bytes each: lbo = bytes between the two core matrices of one MMA along K, sbo = bytes between core matrices
// that are adjacent along M.  Layout type 0 = SWIZZLE_NONE ("interleave").
__device__ __forceinline__ uint64_t umma_desc_cores(uint32_t smem_addr, uint32_t lbo, uint32_t sbo) {
  uint64_t desc = 0;
  desc |= (uint64_t)((smem_addr >> 4) & 0x3fffu);
  desc |= (uint64_t)((lbo >> 4) & 0x3fffu) << 16;
  desc |= (uint64_t)((sbo >> 4) & 0x3fffu) << 32;
  desc |= (uint64_t)1 << 46;                                 // version
  return desc;
}
// Instruction descriptor: D fp32, A and B bf16, both K-major, M x N tile.
__device__ __forceinline__ uint32_t umma_idesc_bf16(int M, int N) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}

// Work list of one wave: one item per (wave entry, tile of kMmaNT routed pairs), resolved: work4[w] = (first sorted pair
// position, valid pairs, slot, plan entry index); *n_work = item count.  One warp.
__global__ void __launch_bounds__(32) build_work_kernel(PlanPtrs plan, int wave, int C, int* __restrict__ work, int* __restrict__ n_work) {
  const int lane = threadIdx.x;
  int n = 0;
  if (wave < plan.hdr[0]) {
    const int lo = wave * C, hi = min(plan.hdr[1], lo + C);
    for (int i0 = lo; i0 < hi; i0 += 32) {                    // 32 entries at a time: tile counts, warp prefix sum, scatter
      const int i = i0 + lane;
      const int e = i < hi ? plan.entry_expert[i] : 0;
      const int cnt = i < hi ? plan.exp_count[e] : 0;
      const int off = i < hi ? plan.exp_offset[e] : 0, slot = i < hi ? plan.entry_slot[i] : 0;
      const int tiles = (cnt + kMmaNT - 1) / kMmaNT;
      int inc = tiles;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += v; }
      int pos = n + inc - tiles;
      for (int p0 = 0; p0 < cnt; p0 += kMmaNT, ++pos)
        reinterpret_cast<int4*>(work)[pos] = make_int4(off + p0, min(kMmaNT, cnt - p0), slot, i);
      n += __shfl_sync(0xffffffffu, inc, 31);
    }
  }
  if (lane == 0) *n_work = n;
}

// Persistent: one CTA per SM walks the tiles t = blockIdx.x, blockIdx.x + gridDim.x, ...; tile t = (work item t / RT,
// 128-row tile t % RT) with RT = weight rows / 128.  Two TMEM accumulator stages: the epilogue of tile j drains
// stage j & 1 while the MMA warp already fills the other stage with tile j + 1.
// tm_w: 3-D map over the arena (K, weight row, blob); tm_x: 2-D map over the B rows (K, sorted pair position).
template <int MODE>
__global__ void __launch_bounds__(kMmaThreads, 1) prefill_mma_kernel(const __grid_constant__ CUtensorMap tm_w,
                                                                     const __grid_constant__ CUtensorMap tm_x,
                                                                     const MmaArgs a, const int* __restrict__ work,
                                                                     const int* __restrict__ n_work_p, const int n_stages) {
  extern __shared__ __align__(1024) unsigned char smem_mma[];
  __shared__ __align__(8) unsigned long long s_full[8], s_empty[8], s_tfull[2], s_tempty[2];
  __shared__ uint32_t s_tmem;
  // weight tiles per stage: gate + up | two 128-row blocks of down (they share the B tile: the kernels run at the L2->SM rate
  // of the TMA path, ~12 TB/s chip-wide, so every B re-read that is avoided is time) | router rows
  constexpr int NA = MODE == 2 ? 1 : 2;
  constexpr uint32_t kStage = (NA + 1) * kMmaTileBytes;
  const uint32_t stage_tx = MODE == 2 ? NA * kMmaTileBytes + (uint32_t)a.b_rows * (kMmaBK * 2) : kStage;   // bytes a stage receives
  constexpr uint32_t kAccCols = MODE == 2 ? 128 : 256;        // TMEM columns of one accumulator stage
  constexpr uint32_t kCols = 2 * kAccCols;

  const int K = MODE == 1 ? a.dff : a.d;
  const int nkb = K / kMmaBK;
  const int RT = MODE == 0 ? a.dff / kMmaM : MODE == 1 ? a.d / (2 * kMmaM) : a.E / kMmaM;
  const int n_tiles = (MODE == 2 ? (a.n_tokens + a.b_rows - 1) / a.b_rows : *n_work_p) * RT;
  if ((int)blockIdx.x >= n_tiles) return;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t smem0 = (smem_u32(smem_mma) + 1023u) & ~1023u;   // swizzle-128B tiles need 1024-byte alignment
  if (tid == 0) {
    for (int s = 0; s < n_stages; ++s) { mbar_init(smem_u32(&s_full[s]), 1); mbar_init(smem_u32(&s_empty[s]), 1); }
    for (int s = 0; s < 2; ++s) { mbar_init(smem_u32(&s_tfull[s]), 1); mbar_init(smem_u32(&s_tempty[s]), 4); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 1) tmem_alloc(smem_u32(&s_tmem), kCols);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = s_tmem;

  if (warp == 0) {
    if (lane == 0) {      // ===== TMA producer =====
      int s = 0; uint32_t ph = 0;
      MmaTile nxt = mma_tile<MODE>(a, work, blockIdx.x, RT);
      for (int t = blockIdx.x; t < n_tiles; t += gridDim.x) {
        const MmaTile mt = nxt;
        if (t + (int)gridDim.x < n_tiles) nxt = mma_tile<MODE>(a, work, t + gridDim.x, RT);   // in flight while this tile streams
        const int r0 = mt.r0, pos0 = mt.pos0, blob = mt.blob;
        for (int kb = 0; kb < nkb; ++kb) {
          mbar_wait(smem_u32(&s_empty[s]), ph ^ 1u);
          const uint32_t bar = smem_u32(&s_full[s]);
          mbar_expect_tx(bar, stage_tx);
          const uint32_t base = smem0 + s * kStage;
          if (MODE == 0) {          // (core, core column = K block, core row = row group, blob): gate then up
            tma_load_4d(base, &tm_w, 0, kb * (kMmaBK / 8), r0 / 8, blob, bar);
            tma_load_4d(base + kMmaTileBytes, &tm_w, 0, kb * (kMmaBK / 8), (a.dff + r0) / 8, blob, bar);
          } else if (MODE == 1) {   // (core, output group j/8, act-column block i/8, blob)
            tma_load_4d(base, &tm_w, 0, r0 / 8, kb * (kMmaBK / 8), blob, bar);
            tma_load_4d(base + kMmaTileBytes, &tm_w, 0, (r0 + kMmaM) / 8, kb * (kMmaBK / 8), blob, bar);
          } else {
            tma_load_3d(base, &tm_w, kb * kMmaBK, r0, blob, bar);
          }
          tma_load_2d(base + NA * kMmaTileBytes, &tm_x, kb * kMmaBK, pos0, bar);
          if (++s == n_stages) { s = 0; ph ^= 1u; }
        }
      }
    }
  } else if (warp == 1) {
    if (lane == 0) {      // ===== MMA issuer =====
      int s = 0; uint32_t ph = 0;
      int j = 0;
      int nt_next = mma_tile<MODE>(a, work, blockIdx.x, RT).nt;
      for (int t = blockIdx.x; t < n_tiles; t += gridDim.x, ++j) {
        const int nt = nt_next;
        if (t + (int)gridDim.x < n_tiles) nt_next = mma_tile<MODE>(a, work, t + gridDim.x, RT).nt;
        const uint32_t idesc = umma_idesc_bf16(kMmaM, max(16, (nt + 15) & ~15));
        const int as = j & 1;
        mbar_wait(smem_u32(&s_tempty[as]), ((uint32_t)(j >> 1) & 1u) ^ 1u);   // the epilogue has drained this stage
        tc_fence_after();
        const uint32_t acc_base = tmem + as * kAccCols;
        for (int kb = 0; kb < nkb; ++kb) {
          mbar_wait(smem_u32(&s_full[s]), ph);
          tc_fence_after();
          const uint32_t base = smem0 + s * kStage;
          // A: MODE 0 tile = [16 row groups][8 K cores][128 B]  (K-adjacent cores 128 B apart, row groups 1 KiB apart; 16 K
          //                   elements = 2 cores = 256 B per MMA);
          //    MODE 1 tile = [8 K blocks][16 output groups][128 B] (K-adjacent cores 2 KiB apart, output groups 128 B apart;
          //                   4 KiB per MMA);  MODE 2 (router rows, row-major in global memory) = 128-byte swizzle
          const uint64_t da0 = MODE == 0 ? umma_desc_cores(base, 128u, 1024u) : MODE == 1 ? umma_desc_cores(base, 2048u, 128u) : umma_desc_sw128(base);
          const uint64_t da1 = MODE == 1 ? umma_desc_cores(base + kMmaTileBytes, 2048u, 128u) : umma_desc_cores(base + kMmaTileBytes, 128u, 1024u);
          const uint32_t a_step = MODE == 0 ? 256u >> 4 : MODE == 1 ? 4096u >> 4 : 2u;
          const uint64_t db = umma_desc_sw128(base + NA * kMmaTileBytes);
#pragma unroll
          for (int k4 = 0; k4 < kMmaBK / 16; ++k4) {          // UMMA_K = 16 bf16
            const uint32_t acc = (kb | k4) != 0;
            umma_bf16(acc_base, da0 + a_step * k4, db + 2 * k4, idesc, acc);
            if (MODE != 2) umma_bf16(acc_base + 128, da1 + a_step * k4, db + 2 * k4, idesc, acc);
          }
          umma_commit(smem_u32(&s_empty[s]));                 // frees the stage once these MMAs have read it
          if (++s == n_stages) { s = 0; ph ^= 1u; }
        }
        umma_commit(smem_u32(&s_tfull[as]));                  // accumulators of this tile complete
      }
    }
  } else {                // ===== epilogue warps: TMEM lane quarter = warp % 4 =====
    const int q = warp & 3;
    int j = 0;
    MmaTile nxt = mma_tile<MODE>(a, work, blockIdx.x, RT);
    for (int t = blockIdx.x; t < n_tiles; t += gridDim.x, ++j) {
      const MmaTile mt = nxt;
      if (t + (int)gridDim.x < n_tiles) nxt = mma_tile<MODE>(a, work, t + gridDim.x, RT);
      const int r0 = mt.r0, pos0 = mt.pos0, nt = mt.nt;
      const int N = max(16, (nt + 15) & ~15);
      const int as = j & 1;
      mbar_wait(smem_u32(&s_tfull[as]), (uint32_t)(j >> 1) & 1u);
      tc_fence_after();
      const int row = r0 + 32 * q + lane;                     // weight row = d_ff index (MODE 0) | d index (MODE 1; second block: + 128)
      const uint32_t tlane = tmem + as * kAccCols + ((uint32_t)(32 * q) << 16);
      const int* pl = MODE == 2 ? nullptr : a.plan.pair_list + pos0;
      const float bias_r = MODE == 2 ? a.bias[row] : 0.f;
      for (int c0 = 0; c0 < N; c0 += 16) {
        float g[16], u[16];
        // MODE 1: the pair ids of these 16 columns in ONE load (lane l holds column c0 + l % 16), handed round by shuffles --
        // a dependent global load per column was half of this warp's time
        int my_pair = 0;
        if (MODE == 1) my_pair = pl[min(c0 + (lane & 15), nt - 1)];
        tmem_ld16(tlane + c0, g);
        if (MODE != 2) tmem_ld16(tlane + 128 + c0, u);
#pragma unroll
        for (int jj = 0; jj < 16; ++jj) {
          const int col = c0 + jj;
          const int pr = MODE == 1 ? __shfl_sync(0xffffffffu, my_pair, jj) : 0;
          if (col < nt) {
            if (MODE == 0) a.act[(size_t)(pos0 + col) * a.dff + row] = __float2bfloat16_rn(silu_f(g[jj]) * u[jj]);
            else if (MODE == 1) { a.ystage[(size_t)pr * a.d + row] = g[jj]; a.ystage[(size_t)pr * a.d + row + kMmaM] = u[jj]; }
            else a.z[(size_t)(pos0 + col) * a.E + row] = g[jj] + bias_r;
          }
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(smem_u32(&s_tempty[as]));    // this warp's quarter of the stage is drained
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) tmem_dealloc(tmem, kCols);
}

// xg[pos][:] = x[pair_list[pos] / k][:] for every routed pair (sorted by expert): the B operand of GEMM 1.  One warp per pair and
// iteration, the row's 16-byte pieces of a lane loaded before any is stored (8 CTAs x 8 warps per SM keep the copies in flight).
__global__ void __launch_bounds__(256) gather_tokens_kernel(const int* __restrict__ pair_list, int n_pairs, int k, int d_vec,
                                                            const uint4* __restrict__ x, uint4* __restrict__ xg) {
  const int lane = threadIdx.x & 31, wpb = blockDim.x >> 5;
  for (int pos = blockIdx.x * wpb + (threadIdx.x >> 5); pos < n_pairs; pos += gridDim.x * wpb) {
    const uint4* src = x + (size_t)(__ldg(pair_list + pos) / k) * d_vec;
    uint4* dst = xg + (size_t)pos * d_vec;
    for (int c0 = lane; c0 < d_vec; c0 += 32 * 8) {
      uint4 v[8];
#pragma unroll
      for (int u = 0; u < 8; ++u) v[u] = __ldg(src + min(c0 + 32 * u, d_vec - 1));
#pragma unroll
      for (int u = 0; u < 8; ++u)
        if (c0 + 32 * u < d_vec) __stcs(dst + c0 + 32 * u, v[u]);
    }
  }
}

}  // namespace wisp
