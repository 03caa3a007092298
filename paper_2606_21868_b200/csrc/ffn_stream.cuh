// ffn_stream.cuh -- (a4) decode expert SwiGLU FFN over slot-indirected weights as HBM-streaming GEMV
// kernels for sm_100a (1 flop/byte: plain ALUs, no tensor cores), with the fused variant of the miss
// path (a3).  The FFN itself is the engine's in the paper ("unmodified fused-MoE kernel",
// PAPER.md:108-110); BASELINE.json fixes SwiGLU (G8, G21):
//   MODE 0 (gate_up): g = W_gate[s] x_t, u = W_up[s] x_t, act = silu(g) * u     (act kept in fp32)
//   MODE 1 (down)   : y = W_down[s] act                                        (y staged in fp32)
// One persistent CTA per SM.  A producer warp streams the wave's weight tiles through a shared-memory
// ring with 1-D TMA bulk copies (cp.async.bulk + mbarrier complete_tx); 8 consumer warps hold a
// thread-stationary K-slice of the operand (x or act) in registers, FMA against the tile and reduce.
//
// Work decomposition:
//   segment  = seg_chunks 16-byte chunks of one weight row (seg_chunks = P <= 256 threads, one chunk each)
//   stage    = RB rows x n_mats matrices x one segment  (<= 32 KiB)      -> one ring slot
//   unit     = (wave entry, row block of RB rows), all NSEG segments      -> one reduction + epilogue
//   CTA c takes the contiguous unit range [c*U/grid, (c+1)*U/grid).
// Canonical summation order of every (row, pair) dot product (parity (b)): thread p
// accumulates elements of chunk p of segment 0, 1, ... in ascending order with fmaf into one fp32
// accumulator; the P/32 warps' lanes are combined by an xor butterfly (16, 8, 4, 2, 1); the warp sums are
// added in ascending warp order.  Nothing in it depends on the slot, the wave, the CTA, the number of
// tokens in the call or whether the tile came from HBM or from the host master.
//
// Fused miss path (WISP_FETCH_FUSED): for an entry that the residency step marked as a miss, the producer
// reads the tile from the mapped pinned host master (Alg. 1 line 6) instead of the slot,
// and consumer warp 0 writes the landed tile from shared memory into the victim slot with a bulk store.
// The FFN consumes the same bytes in the same order as on a hit, so outputs are byte-identical.
#pragma once
#include "common.cuh"

namespace wisp {

constexpr int kStreamConsumers = 256;                       // 8 consumer warps
constexpr int kStreamThreads = kStreamConsumers + 32;       // + 1 producer warp
constexpr int kStreamMaxStages = 8;
// Weight rows per consumer thread per ring stage: 16 (8 gate + 8 up | 16 down; 64 KiB stages) when at most 2 tokens are in
// flight, 8 (32 KiB stages) otherwise.  Measured on B200 at the Qwen3 shape: 64 KiB stages x 2 beat 32 KiB x 3 by 5 % at batch 1
// (larger TMA copies), but at batch 4 their 64 accumulators per thread spill.  The geometry (StreamGeom.RB) follows the same rule.
template <int NP> struct StreamVals { static constexpr int V = NP <= 2 ? 16 : 8; };
__host__ __device__ constexpr int stream_vals_for_tokens(int n_tokens) { return n_tokens <= 2 ? 16 : 8; }

__device__ __forceinline__ float silu_f(float v) { return v / (1.0f + expf(-v)); }

// ---- PTX wrappers: mbarrier, TMA bulk copies, programmatic dependent launch ---------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "LAB_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
      "@P1 bra DONE;\n"
      "bra LAB_WAIT;\n"
      "DONE:\n"
      "}" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ uint64_t l2_evict_first_policy() {
  uint64_t p;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
  return p;
}
// global -> shared bulk copy, completion signalled on `bar` (SASS: UBLKCP)
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar, uint64_t policy) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(dst),
               "l"(src), "r"(bytes), "r"(bar), "l"(policy) : "memory");
}
__device__ __forceinline__ void bulk_g2s_nohint(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src), "r"(bytes),
               "r"(bar) : "memory");
}
// shared -> global bulk copy (bulk async-group)
__device__ __forceinline__ void bulk_s2g(void* dst, uint32_t src, uint32_t bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait0() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// ---- geometry (computed on the host once per context) ---------------------------------------------------
struct StreamGeom {
  int K;                 // reduction length in elements (d_model for gate/up, d_ff for down)
  int rows;              // rows per matrix (d_ff | d_model)
  int n_mats;            // 2 (gate, up) | 1 (down)
  unsigned long long mat_off[2];   // byte offset of each matrix inside the expert blob
  int row_bytes;         // K * sizeof(T)
  int P;                 // threads per row group = chunks per segment
  int G;                 // row groups per CTA (G * P <= 256)
  int RB;                // rows per matrix per stage = (vals / n_mats) * G
  int NSEG;              // segments per row
  int seg_bytes;         // P * 16
  int stage_bytes;       // n_mats * RB * seg_bytes
  int upe;               // units per entry = rows / RB
  int n_active;          // G * P consumer threads that do work
  int n_stages;          // ring depth
};

struct StreamArgs {
  PlanPtrs plan;
  int wave, C;
  const char* pool;      // arena base; slot s of layer l at ((size_t)s * L + l) * blob_bytes
  const char* master;    // mapped pinned host master of this layer (E blobs) or nullptr (no fused fill)
  unsigned long long blob_bytes;
  int L, layer;
  const void* operand;   // MODE 0: x [T, d] model dtype; MODE 1: act [T*k, d_ff] fp32
  float* result;         // MODE 0: act [T*k, d_ff] fp32; MODE 1: ystage [T*k, d] fp32
  int k;                 // top_k (pair index = t*k + rank)
  int out_ld;            // leading dimension of result (d_ff | d)
  int pdl;               // launched with programmatic stream serialization
};

// Transposed butterfly: reduces NV per-lane values over the 32 lanes with NV-1 (+ log) shuffles.  The sum
// of value i ends up in v[j] of lane L with (L*NV)/32 + j == i (j < max(1, NV/32)); for every value the
// addition tree is the xor butterfly 16, 8, 4, 2, 1 (fp add commutes, so all lanes agree bit for bit).
template <int NV>
__device__ __forceinline__ void warp_multi_reduce(float (&v)[NV], int lane) {
  int n = NV;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const bool up = (lane & o) != 0;
    if (n > 1) {
      const int h = n >> 1;
#pragma unroll
      for (int i = 0; i < NV / 2; ++i) {
        if (i < h) {
          const float keep = up ? v[i + h] : v[i];
          const float send = up ? v[i] : v[i + h];
          v[i] = keep + __shfl_xor_sync(0xffffffffu, send, o);
        }
      }
      n = h;
    } else {
      v[0] += __shfl_xor_sync(0xffffffffu, v[0], o);
    }
  }
}

// ---- the shared-memory ring ------------------------------------------------------------------------------
struct Ring {
  uint32_t stage0;         // shared address of stage 0
  uint32_t full0, empty0;  // shared addresses of the full / empty mbarrier arrays (8 bytes per stage)
  int NS;                  // stages in use
  int stride;              // bytes between stages (>= the stage_bytes of every geometry that uses the ring)
};
struct RingPos { int s; uint32_t ph; };
__device__ __forceinline__ void ring_advance(const Ring& r, RingPos& p) { if (++p.s == r.NS) { p.s = 0; p.ph ^= 1u; } }
// full barriers: 1 arrival (the producer's expect_tx); empty barriers: one arrival per consumer warp
__device__ __forceinline__ void ring_init(const Ring& r) {
  for (int s = 0; s < r.NS; ++s) {
    mbar_init(r.full0 + 8u * s, 1);
    mbar_init(r.empty0 + 8u * s, kStreamConsumers / 32);
  }
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}

// Units [u_lo, u_hi) of the wave whose first plan entry is `lo`: the producer warp issues the TMA bulk loads.
__device__ __forceinline__ void stream_produce(const StreamArgs& a, const StreamGeom& gm, const Ring& ring, RingPos& rp,
                                               int lo, int u_lo, int u_hi, int lane, uint64_t pol) {
  const int n_copies = gm.NSEG == 1 ? gm.n_mats : gm.n_mats * gm.RB;
  for (int u = u_lo; u < u_hi; ++u) {
    const int i = lo + u / gm.upe, rb = u % gm.upe;
    const bool from_host = a.master != nullptr && a.plan.entry_miss[i] != 0;
    const char* blob = from_host ? a.master + (size_t)a.plan.entry_expert[i] * a.blob_bytes
                                 : a.pool + ((size_t)a.plan.entry_slot[i] * a.L + a.layer) * a.blob_bytes;
    for (int seg = 0; seg < gm.NSEG; ++seg) {
      mbar_wait(ring.empty0 + 8u * rp.s, rp.ph ^ 1u);
      const uint32_t bar = ring.full0 + 8u * rp.s;
      if (lane == 0) mbar_expect_tx(bar, (uint32_t)gm.stage_bytes);
      __syncwarp();
      const uint32_t sbase = ring.stage0 + (uint32_t)rp.s * ring.stride;
      for (int c = lane; c < n_copies; c += 32) {
        const char* src;
        uint32_t bytes;
        if (gm.NSEG == 1) {        // the RB rows of one matrix are contiguous: one copy per matrix
          bytes = (uint32_t)gm.RB * gm.row_bytes;
          src = blob + gm.mat_off[c] + (size_t)rb * gm.RB * gm.row_bytes;
        } else {                   // one copy per (matrix, row): a seg_bytes slice of the row
          const int m = c / gm.RB, r = c % gm.RB;
          bytes = (uint32_t)gm.seg_bytes;
          src = blob + gm.mat_off[m] + ((size_t)rb * gm.RB + r) * gm.row_bytes + (size_t)seg * gm.seg_bytes;
        }
#ifdef WISP_PROBE_NO_L2_HINT   // profiling probe only
        bulk_g2s_nohint(sbase + c * bytes, src, bytes, bar);
#else
        bulk_g2s(sbase + c * bytes, src, bytes, bar, pol);
#endif
      }
      ring_advance(ring, rp);
    }
  }
}

// Accumulators per consumer thread between two reductions: 32 (64 for 8 pairs) = row blocks per batch x 8 rows x CNT,
// CNT = routed pairs of the expert rounded up to 1, 2, 4 or 8.  The shared-memory scratch is sized for the kernel's NP.
template <int CNT, int V> struct StreamBatch {
  static constexpr int SPU = (32 / V) / CNT > 0 ? (32 / V) / CNT : 1;   // row blocks (ring stages per segment) per batch
  static constexpr int NVAL = SPU * V * CNT;                // values reduced per thread per batch
};
__device__ __forceinline__ int stream_cnt_class(int cnt) { return cnt <= 1 ? 1 : cnt <= 2 ? 2 : cnt <= 4 ? 4 : 8; }

// Row blocks [u, u_end) of ONE plan entry i (all inside this CTA's unit range), pairs pl[0..cnt), cnt <= CNT.
// Thread p of a row group keeps chunk p of each pair's operand in registers and one fp32 accumulator per (row, pair);
// up to SPU consecutive row blocks are accumulated before ONE cross-thread reduction (lanes: transposed xor butterfly;
// warps: ascending, through s_red) and one epilogue, so the block-wide barrier and the SiLU/store tail are paid once
// per batch, not once per ring stage.  Batching changes which dot products are reduced together, never the summation
// order inside one of them; an unused pair slot (cnt < CNT) multiplies by a zero operand and is never stored.
template <typename T, int MODE, int CNT, int V>
__device__ __forceinline__ void stream_consume_entry(const StreamArgs& a, const StreamGeom& gm, const Ring& ring, RingPos& rp,
                                                     int i, int u, int u_end, int cnt, const int* pl, float* s_red, int& par,
                                                     int red_bar) {
  constexpr int EPC = ChunkW<T>::N;                         // elements per 16-byte chunk
  constexpr int kStreamVals = V;
  constexpr int SPU = StreamBatch<CNT, V>::SPU;
  constexpr int NVAL = StreamBatch<CNT, V>::NVAL;
  constexpr int RPT = kStreamVals / (MODE == 0 ? 2 : 1);    // rows per thread per matrix per row block
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid >= gm.n_active) {
    // a warp without work in this geometry still takes part in the ring protocol (the empty barriers count 8 warps)
    while (u < u_end) {
      const int nb = min(SPU, u_end - u);
      for (int j = 0; j < nb * gm.NSEG; ++j) {
        mbar_wait(ring.full0 + 8u * rp.s, rp.ph);
        if (lane == 0) mbar_arrive(ring.empty0 + 8u * rp.s);
        ring_advance(ring, rp);
      }
      u += nb;
      par ^= 1;                     // stay in step with the active warps' s_red half: one flip per batch
    }
    return;
  }
  const int g = tid / gm.P, p = tid % gm.P;
  const int warps_per_group = gm.P >> 5;
  const bool fill = a.master != nullptr && a.plan.entry_miss[i] != 0;
  float xr[CNT][EPC];
  bool need_operand = true;
  while (u < u_end) {
    const int rb0 = u % gm.upe;
    const int nb = min(SPU, u_end - u);                     // row blocks of this batch
    float acc[SPU][kStreamVals][CNT];
#pragma unroll
    for (int b = 0; b < SPU; ++b)
#pragma unroll
      for (int v = 0; v < kStreamVals; ++v)
#pragma unroll
        for (int q = 0; q < CNT; ++q) acc[b][v][q] = 0.f;
#pragma unroll
    for (int b = 0; b < SPU; ++b) {
      if (b < nb) {
        const int rb = rb0 + b;
        for (int seg = 0; seg < gm.NSEG; ++seg) {
          if (need_operand || gm.NSEG > 1) {    // (re)load the thread-stationary operand slice
#pragma unroll
            for (int q = 0; q < CNT; ++q) {
              if (q < cnt) {
                const int pr = pl[q];
                const size_t col = (size_t)seg * gm.P * EPC + (size_t)p * EPC;
                if (MODE == 0) {
                  const T* xp = reinterpret_cast<const T*>(a.operand) + (size_t)(pr / a.k) * gm.K + col;
                  ChunkW<T>::widen(*reinterpret_cast<const uint4*>(xp), xr[q]);
                } else {
                  const float* ap = reinterpret_cast<const float*>(a.operand) + (size_t)pr * gm.K + col;
#pragma unroll
                  for (int j = 0; j < EPC; j += 4) {
                    const float4 f = *reinterpret_cast<const float4*>(ap + j);
                    xr[q][j] = f.x; xr[q][j + 1] = f.y; xr[q][j + 2] = f.z; xr[q][j + 3] = f.w;
                  }
                }
              } else {
#pragma unroll
                for (int j = 0; j < EPC; ++j) xr[q][j] = 0.f;
              }
            }
            need_operand = false;
          }
          mbar_wait(ring.full0 + 8u * rp.s, rp.ph);
#ifdef WISP_PROBE_SKIP_MATH   // profiling probe only (never built into the product): the ring's pure streaming rate
          __syncwarp();
          if (lane == 0) mbar_arrive(ring.empty0 + 8u * rp.s);
          ring_advance(ring, rp);
          continue;
#endif
          const uint32_t sbase = ring.stage0 + (uint32_t)rp.s * ring.stride;
          if (fill && warp == 0) {           // fused miss path: landed tile -> victim slot (same bytes)
            char* slot = const_cast<char*>(a.pool) + ((size_t)a.plan.entry_slot[i] * a.L + a.layer) * a.blob_bytes;
            const int n_copies = gm.NSEG == 1 ? gm.n_mats : gm.n_mats * gm.RB;
            for (int c = lane; c < n_copies; c += 32) {
              if (gm.NSEG == 1) {
                const uint32_t bytes = (uint32_t)gm.RB * gm.row_bytes;
                bulk_s2g(slot + gm.mat_off[c] + (size_t)rb * gm.RB * gm.row_bytes, sbase + c * bytes, bytes);
              } else {
                const int m = c / gm.RB, r = c % gm.RB;
                bulk_s2g(slot + gm.mat_off[m] + ((size_t)rb * gm.RB + r) * gm.row_bytes + (size_t)seg * gm.seg_bytes,
                         sbase + c * gm.seg_bytes, (uint32_t)gm.seg_bytes);
              }
            }
            bulk_commit();
          }
          if constexpr (CNT <= 2) {
            // this thread's 8 weight chunks of the stage: matrix m, row g*RPT + i, chunk p; the stage is released as
            // soon as they are in registers
            uint4 wq[kStreamVals];
#pragma unroll
            for (int v = 0; v < kStreamVals; ++v) {
              const int m = MODE == 0 ? v / RPT : 0, r = g * RPT + (MODE == 0 ? v % RPT : v);
              const uint32_t addr = sbase + (uint32_t)((m * gm.RB + r) * gm.seg_bytes + p * 16);
              asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(wq[v].x), "=r"(wq[v].y), "=r"(wq[v].z), "=r"(wq[v].w) : "r"(addr));
            }
            if (fill && warp == 0) bulk_wait_read0();   // the bulk store has finished reading the stage
            __syncwarp();
            if (lane == 0) mbar_arrive(ring.empty0 + 8u * rp.s);   // stage free: the data lives in registers now
            ring_advance(ring, rp);
#pragma unroll
            for (int v = 0; v < kStreamVals; ++v) {
              float wv[EPC];
              ChunkW<T>::widen(wq[v], wv);
#pragma unroll
              for (int q = 0; q < CNT; ++q)
#pragma unroll
                for (int j = 0; j < EPC; ++j) acc[b][v][q] = fmaf(wv[j], xr[q][j], acc[b][v][q]);
            }
          } else {
            // 4 or 8 pairs: operands and accumulators already fill the register file, so the weight chunks are taken
            // from shared memory one at a time and the stage is released after the last one (same FMA order)
#pragma unroll
            for (int v = 0; v < kStreamVals; ++v) {
              const int m = MODE == 0 ? v / RPT : 0, r = g * RPT + (MODE == 0 ? v % RPT : v);
              const uint32_t addr = sbase + (uint32_t)((m * gm.RB + r) * gm.seg_bytes + p * 16);
              uint4 w1;
              asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(w1.x), "=r"(w1.y), "=r"(w1.z), "=r"(w1.w) : "r"(addr));
              float wv[EPC];
              ChunkW<T>::widen(w1, wv);
#pragma unroll
              for (int q = 0; q < CNT; ++q)
#pragma unroll
                for (int j = 0; j < EPC; ++j) acc[b][v][q] = fmaf(wv[j], xr[q][j], acc[b][v][q]);
            }
            if (fill && warp == 0) bulk_wait_read0();
            __syncwarp();
            if (lane == 0) mbar_arrive(ring.empty0 + 8u * rp.s);
            ring_advance(ring, rp);
          }
        }
      }
    }
#ifndef WISP_PROBE_SKIP_MATH
    // ---- reduce over the group's P threads: lanes (butterfly), then warps (ascending) ----
    float red[NVAL];
#pragma unroll
    for (int b = 0; b < SPU; ++b)
#pragma unroll
      for (int v = 0; v < kStreamVals; ++v)
#pragma unroll
        for (int q = 0; q < CNT; ++q) red[(b * kStreamVals + v) * CNT + q] = acc[b][v][q];
    warp_multi_reduce<NVAL>(red, lane);
    constexpr int PER_LANE = NVAL >= 32 ? NVAL / 32 : 1;
    float* sr = s_red + (size_t)par * (kStreamConsumers / 32) * NVAL;
#pragma unroll
    for (int j = 0; j < PER_LANE; ++j) sr[warp * NVAL + (lane * NVAL) / 32 + j] = red[j];
    asm volatile("bar.sync %0, %1;" ::"r"(red_bar), "r"(gm.n_active) : "memory");
    const int n_out = nb * gm.RB * cnt;                    // (row block, row inside the block, pair)
    for (int o = tid; o < n_out; o += gm.n_active) {
      const int q = o % cnt, rr = o / cnt;
      const int b = rr / gm.RB, r = rr % gm.RB;
      const int rg = r / RPT, ri = r % RPT;
      const int w0 = (rg * gm.P) >> 5;
      const int pr = pl[q];
      const size_t row = (size_t)(rb0 + b) * gm.RB + r;
      const float* base = sr + (size_t)w0 * NVAL + (b * kStreamVals) * CNT + q;
      if (MODE == 0) {
        float gs = 0.f, us = 0.f;
        for (int w = 0; w < warps_per_group; ++w) {
          gs += base[w * NVAL + ri * CNT];
          us += base[w * NVAL + (RPT + ri) * CNT];
        }
        a.result[(size_t)pr * a.out_ld + row] = silu_f(gs) * us;
      } else {
        float ys = 0.f;
        for (int w = 0; w < warps_per_group; ++w) ys += base[w * NVAL + ri * CNT];
        a.result[(size_t)pr * a.out_ld + row] = ys;
      }
    }
#endif
    par ^= 1;
    u += nb;
  }
}

// The 8 consumer warps (tid 0..255) take units [u_lo, u_hi) of the wave whose first plan entry is `lo` from the ring, entry
// by entry; each entry runs the routine instantiated for its pair count class (1, 2, 4, 8 <= NP), so an expert routed by
// one token of a batch still batches 4 row blocks per reduction.  MODE 0 = gate/up + SwiGLU, MODE 1 = down.
// s_red: [2][8][StreamBatch<NP>::NVAL-or-32] floats of shared memory; `par` alternates between its halves; `red_bar` = a
// named barrier id free for the n_active threads.
template <typename T, int MODE, int NP>
__device__ __forceinline__ void stream_consume(const StreamArgs& a, const StreamGeom& gm, const Ring& ring, RingPos& rp,
                                               int lo, int u_lo, int u_hi, float* s_red, int& par, int red_bar) {
  for (int u = u_lo; u < u_hi;) {
    const int i = lo + u / gm.upe;
    const int u_end = min(u_hi, (u / gm.upe + 1) * gm.upe);            // this entry's row blocks inside the range
    const int e = a.plan.entry_expert[i];
    const int cnt = min(a.plan.exp_count[e], NP);
    const int* pl = a.plan.pair_list + a.plan.exp_offset[e];
    const int cls = stream_cnt_class(cnt);
    if (NP == 1 || cls == 1) stream_consume_entry<T, MODE, 1, StreamVals<NP>::V>(a, gm, ring, rp, i, u, u_end, cnt, pl, s_red, par, red_bar);
    else if (NP == 2 || cls == 2) stream_consume_entry<T, MODE, (NP >= 2 ? 2 : 1), StreamVals<NP>::V>(a, gm, ring, rp, i, u, u_end, cnt, pl, s_red, par, red_bar);
    else if (NP == 4 || cls == 4) stream_consume_entry<T, MODE, (NP >= 4 ? 4 : 1), StreamVals<NP>::V>(a, gm, ring, rp, i, u, u_end, cnt, pl, s_red, par, red_bar);
    else stream_consume_entry<T, MODE, (NP >= 8 ? 8 : 1), StreamVals<NP>::V>(a, gm, ring, rp, i, u, u_end, cnt, pl, s_red, par, red_bar);
    u = u_end;
  }
  if (a.master != nullptr && threadIdx.x < 32) bulk_wait0();   // warp 0's slot writes are complete
}

// shared-memory floats of s_red for a kernel instantiated for NP pairs: two halves x 8 warps x the largest batch
template <int NP> struct StreamRed { static constexpr int kFloats = 2 * (kStreamConsumers / 32) * (NP >= 8 ? 64 : 32); };

// One wave of one FFN half as its own launch (multi-kernel path: MEMCPY / ZEROCOPY contexts, timing level 2).
template <typename T, int MODE, int NP>
__global__ void __launch_bounds__(kStreamThreads, 1) ffn_stream_kernel(const StreamArgs a, const StreamGeom gm) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  __shared__ __align__(8) unsigned long long s_full[kStreamMaxStages], s_empty[kStreamMaxStages];
  __shared__ float s_red[StreamRed<NP>::kFloats];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  Ring ring;
  ring.stage0 = smem_u32(smem_raw); ring.full0 = smem_u32(s_full); ring.empty0 = smem_u32(s_empty);
  ring.NS = gm.n_stages; ring.stride = gm.stage_bytes;
  if (tid == 0) ring_init(ring);
  __syncthreads();
  if (a.pdl) {
    // Everything this kernel reads was written by preceding kernels.  The down producer is exempt: the plan
    // dates from before the gate/up kernel's own wait and down weights are never written by that kernel, so it
    // starts streaming while the gate/up kernel (the immediate predecessor) drains.
    if (MODE == 0 || warp != kStreamConsumers / 32) pdl_wait();
    pdl_launch_dependents();          // the next kernel may start its prologue as SMs drain
  }
  if (a.wave >= a.plan.hdr[0]) return;
  const int lo = a.wave * a.C, nw = min(a.plan.hdr[1], lo + a.C) - lo;
  const long long U = (long long)nw * gm.upe;
  const int u_lo = (int)(U * blockIdx.x / gridDim.x), u_hi = (int)(U * (blockIdx.x + 1) / gridDim.x);
  if (u_lo >= u_hi) return;
  RingPos rp{0, 0u};
  if (warp == kStreamConsumers / 32) {
    stream_produce(a, gm, ring, rp, lo, u_lo, u_hi, lane, l2_evict_first_policy());
  } else {
    int par = 0;
    stream_consume<T, MODE, NP>(a, gm, ring, rp, lo, u_lo, u_hi, s_red, par, 1);
  }
}

// out[t, j] = sum_i w[t,i] * ystage[t*k+i, j] in rank order (fp32), stored in the model dtype; the optional
// residual successor x_next = x + out uses the rounding of DESIGN.md O3.  One function so that the fused
// (router prologue) and the standalone combine produce the same bits.
template <typename T>
__device__ __forceinline__ void combine_elem(const float* ystage, const float* w, int t, int j, int d, int k,
                                             T x_in, T& out, T& x_next) {
  float acc = 0.f;
  for (int i = 0; i < k; ++i) acc = fmaf(w[(size_t)t * k + i], ystage[((size_t)t * k + i) * d + j], acc);
  out = from_f32<T>(acc);
  x_next = from_f32<T>(to_f32<T>(x_in) + to_f32<T>(out));
}

template <typename T>
__global__ void __launch_bounds__(256) combine_kernel(const float* __restrict__ ystage, const float* __restrict__ w,
                                                      T* __restrict__ out, const T* __restrict__ x_res,
                                                      T* __restrict__ x_next, int n_tokens, int d, int k, int pdl) {
  if (pdl) { pdl_wait(); pdl_launch_dependents(); }
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (size_t)n_tokens * d) return;
  const int t = (int)(idx / d), j = (int)(idx % d);
  T o, xn;
  combine_elem<T>(ystage, w, t, j, d, k, x_res ? x_res[idx] : from_f32<T>(0.f), o, xn);
  out[idx] = o;
  if (x_res) x_next[idx] = xn;
}

template <typename T>
__global__ void __launch_bounds__(256) residual_add_kernel(const T* __restrict__ x, const T* __restrict__ y,
                                                           T* __restrict__ out, size_t n) {
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx < n) out[idx] = from_f32<T>(to_f32<T>(x[idx]) + to_f32<T>(y[idx]));
}

}  // namespace wisp
