// decode_ffn.cuh -- (a4) decode expert SwiGLU FFN over slot-indirected weights, fused gate/up/SiLU/down per work unit,
// streaming the weights once from HBM (or, for a missing expert, once over the host link: the fused variant of a3).
// The FFN is the engine's in the paper ("unmodified fused-MoE kernel"); BASELINE.json fixes SwiGLU (G8).
//
// Work unit = (plan entry q = one routed expert, chunk c of RC consecutive act rows i): with the tiled in-slot layout
// (common.cuh) its gate rows, up rows and down COLUMNS are three contiguous pieces, so one CTA computes, without any
// grid-wide exchange in between,
//     g_i = <G[i], x_t>, u_i = <U[i], x_t>, a_i = silu(g_i) * u_i            for the RC rows i of the chunk
//     P[pair][c][j] = sum_{i in chunk} a_i * D[j][i]                          for all j in 0..d-1 (a partial of y)
// for every token routed to the expert (at most 8 tokens per call).  The combine step (decode_combine.cuh) adds the
// chunk partials of an expert in ascending chunk order and the experts of a token in rank order, so
//     y_{t,e}[j] = sum_c P[(t,e)][c][j]   and   out_t = sum_i w[t,i] * y_{t,ids[t,i]}
// have ONE summation order that depends only on the shapes and RC -- not on the slot, the wave, the CTA that happened
// to take the unit, the pool size or hit-vs-miss (parity (b)).  That is what allows the units to be
// handed out DYNAMICALLY (one atomic ticket per unit): the two dies of a B200 stream at different rates and a static
// split leaves the faster one idle at the barrier.
//
// Data path per CTA (288 threads): a producer warp takes tickets and streams each unit's parts (8 rows x one slab of at most
// 32 KiB) through a shared-memory ring with 1-D TMA bulk copies (cp.async.bulk + mbarrier complete_tx); 8 consumer warps
// compute.  bf16: the products run on the tensor cores through mma.sync.m16n8k16 (the 8 MMA columns are the tokens routed
// to the expert; A fragments come straight from the ring with ldmatrix, each core matrix being 128 contiguous bytes), so
// the arithmetic leaves the FMA pipes and the kernel stays a pure HBM stream at 1..8 tokens (1 flop/byte: this is an ALU
// offload of a memory-bound kernel, not a GEMM -- units of 96 KiB are far too small for tcgen05's 128-row tiles).
// fp32 (config 1, parity only): plain FMA with the same data flow and the same reduction tree.
//   gate/up of a sub-block of 8 act rows: warp w owns the K range [w, w+1) * slab/8 of every slab; its 16 x 8 partial tile
//     goes to shared memory, warp 0 adds the 8 warps' partials in ascending warp order, applies SwiGLU, and publishes
//     a[8 rows][8 tokens] (bf16 for bf16 models, G21);
//   down: warp w owns the outputs j in [w, w+1) * slab/8 of every slab and accumulates over the chunk's rows in registers.
// Fused miss path (WISP_FETCH_FUSED): the parts of an entry marked as a miss are read from the mapped pinned master
// (Alg. 1 line 6) and consumer warp 0 stores each landed part into the victim slot with a bulk shared->global
// copy: same bytes, same order of arithmetic as a hit.
#pragma once
#include "common.cuh"

namespace wisp {

constexpr int kDecConsumers = 256;                      // 8 consumer warps
constexpr int kDecWarps = kDecConsumers / 32;
constexpr int kDecThreads = kDecConsumers + 32;         // + 1 producer warp
constexpr int kDecMaxSlots = 8;
constexpr int kDecMaxSteps = 16;                        // MMA steps per warp per part: slab / 128 <= 16
constexpr int kDecUnitQueue = 8;                        // unit ids in flight between producer and consumers
constexpr int kDecMaxPartBytes = 32 << 10;

// Geometry, computed on the host once per context and token class (make_decode_geom in wisp.cu).
struct DecodeGeom {
  int d, dff;
  int elem;              // bytes per weight element
  int kc;                // elements per 16-byte chunk
  int slab;              // elements of d per part (multiple of 256, part_bytes <= 32 KiB)
  int n_slab;            // d / slab
  int part_bytes;        // 8 * slab * elem
  int rows_unit;         // RC: act rows per unit (multiple of 8)
  int n_sb;              // RC / 8 sub-blocks of 8 act rows
  int n_chunks;          // NC = d_ff / RC  (multiple of 8)
  int parts_unit;        // 3 * n_sb * n_slab
  int steps;             // slab / 128
  int down_pieces;       // 8 / kc: bulk copies per down part (the 8 act columns of a sub-block span 8/kc core columns)
  unsigned long long up_off, down_off;    // byte offsets of the up / down matrices inside a blob
  unsigned long long group_bytes;         // 8 * d * elem: one 8-row group of gate/up = the 8 act columns of down
};

struct DecodeFfnArgs {
  const char* pool;       // arena base; slot s of layer l at ((size_t)s * L + l) * blob_bytes
  const char* master;     // mapped pinned master of this layer (fused miss path) or nullptr
  unsigned long long blob_bytes;
  int L, layer, k;
  float* partial;         // P [pair position][NC][d] fp32
  unsigned* ticket;       // unit ticket counter of this wave (zero when the wave starts)
};

// ---- the shared-memory ring -------------------------------------------------------------------------------------
struct DecRing {
  uint32_t slot0;          // shared address of slot 0
  uint32_t full0, empty0;  // shared addresses of the full / empty mbarrier arrays (8 bytes per slot)
  int n_slots;
  int stride;              // bytes between slots
};
struct DecRingPos { int s; uint32_t ph; };
__device__ __forceinline__ void ring_advance(const DecRing& r, DecRingPos& p) { if (++p.s == r.n_slots) { p.s = 0; p.ph ^= 1u; } }
__device__ __forceinline__ void ring_init(const DecRing& r) {   // full: the producer's expect_tx; empty: one arrival per consumer warp
  for (int s = 0; s < r.n_slots; ++s) {
    mbar_init(r.full0 + 8u * s, 1);
    mbar_init(r.empty0 + 8u * s, kDecWarps);
  }
  mbar_fence_init();
}

// Part p of a unit (chunk c): which matrix, sub-block and slab.  Order: every gate/up part first (sub-block major, slab
// minor, gate before up), then the down parts (slab major, sub-block minor) -- so a[] of all sub-blocks exists before the
// first down part and one set of down accumulators serves one slab at a time.
struct DecPart { int mat, sb, slab; };
__device__ __forceinline__ DecPart dec_part(const DecodeGeom& g, int p) {
  DecPart r;
  const int n_gu = 2 * g.n_sb * g.n_slab;
  if (p < n_gu) { r.sb = p / (2 * g.n_slab); const int rem = p % (2 * g.n_slab); r.slab = rem >> 1; r.mat = rem & 1; }
  else { const int q = p - n_gu; r.slab = q / g.n_sb; r.sb = q % g.n_sb; r.mat = 2; }
  return r;
}
// Byte offset inside the blob of piece `piece` of that part.
__device__ __forceinline__ unsigned long long dec_part_offset(const DecodeGeom& g, int c, const DecPart& p, int piece) {
  const unsigned long long grp = (unsigned long long)(c * g.n_sb + p.sb);
  if (p.mat < 2) return (p.mat ? g.up_off : 0ull) + grp * g.group_bytes + (unsigned long long)p.slab * g.part_bytes;
  const unsigned long long pb = (unsigned long long)g.part_bytes / g.down_pieces;
  return g.down_off + (grp * g.down_pieces + piece) * (g.group_bytes / g.down_pieces) + (unsigned long long)p.slab * pb;
}

// ---- producer: one lane takes unit tickets and issues the bulk loads --------------------------------------------
// Units of the wave whose plan entries are [lo, lo + nw): u in [0, nw * NC), entry = unit_entry[lo + u / NC], chunk = u % NC.
// The first unit of CTA b is b (no atomic on the critical path of a phase start), later ones come from the ticket counter.
__device__ __forceinline__ void decode_produce(const DecodeFfnArgs& a, const DecodeGeom& g, const PlanPtrs& plan, const DecRing& ring,
                                               DecRingPos& rp, int& useq, int* s_unit, int lo, int nw, uint64_t pol) {
  const int n_units = nw * g.n_chunks;
  int u = (int)blockIdx.x;
  while (true) {
    if (u >= n_units) {                                        // sentinel: tells the consumers that this wave is over
      mbar_wait(ring.empty0 + 8u * rp.s, rp.ph ^ 1u);
      s_unit[useq & (kDecUnitQueue - 1)] = -1;
      mbar_arrive(ring.full0 + 8u * rp.s);
      ring_advance(ring, rp);
      ++useq;
      return;
    }
    const unsigned t = atomicAdd(a.ticket, 1u);                // next unit: its latency hides behind this unit's copies
    const int q = plan.unit_entry[lo + u / g.n_chunks], c = u % g.n_chunks;
    const bool from_host = a.master != nullptr && plan.entry_miss[q] != 0;
    const char* blob = from_host ? a.master + (size_t)plan.entry_expert[q] * a.blob_bytes
                                 : a.pool + ((size_t)plan.entry_slot[q] * a.L + a.layer) * a.blob_bytes;
    for (int p = 0; p < g.parts_unit; ++p) {
      const DecPart pt = dec_part(g, p);
      mbar_wait(ring.empty0 + 8u * rp.s, rp.ph ^ 1u);
      if (p == 0) s_unit[useq & (kDecUnitQueue - 1)] = u;
      const uint32_t bar = ring.full0 + 8u * rp.s, dst = ring.slot0 + (uint32_t)rp.s * ring.stride;
      mbar_expect_tx(bar, (uint32_t)g.part_bytes);
      const int np = pt.mat == 2 ? g.down_pieces : 1;
      const uint32_t pb = (uint32_t)g.part_bytes / np;
      for (int piece = 0; piece < np; ++piece)
        bulk_g2s(dst + piece * pb, blob + dec_part_offset(g, c, pt, piece), pb, bar, pol);
      ring_advance(ring, rp);
    }
    ++useq;
    u = (int)gridDim.x + (int)t;
  }
}

// C-fragment position of element (row, col) of a 16 x 8 tile inside a warp's 128-float partial (index lane * 4 + reg).
__device__ __forceinline__ int cfrag_index(int row, int col) { return ((row & 7) * 4 + (col >> 1)) * 4 + ((row >> 3) << 1) + (col & 1); }

template <typename T> struct ActT { typedef float type; };
template <> struct ActT<__nv_bfloat16> { typedef __nv_bfloat16 type; };

// ---- consumers: the 8 warps (tid 0..255) process the units the producer queued, until the sentinel ---------------
// xs: the call's hidden states in shared memory, [T][xs_pitch] elements of T (rows padded by 16 bytes).
// s_red: 8 * 128 floats; s_act: 2 * 64 elements of ActT (a[sub-block][token column][act row]).
template <typename T>
__device__ __forceinline__ void decode_consume(const DecodeFfnArgs& a, const DecodeGeom& g, const PlanPtrs& plan, const DecRing& ring,
                                               DecRingPos& rp, int& useq, const int* s_unit, int lo, const T* xs, int xs_pitch,
                                               float* s_red, void* s_act_raw) {
  typedef typename ActT<T>::type AT;
  constexpr bool kMma = sizeof(T) == 2;
  AT* s_act = reinterpret_cast<AT*>(s_act_raw);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int col = lane >> 2, kq = (lane & 3) * 2;             // MMA fragment coordinates of this lane
  while (true) {
    mbar_wait(ring.full0 + 8u * rp.s, rp.ph);
    const int u = s_unit[useq & (kDecUnitQueue - 1)];
    ++useq;
    if (u < 0) {                                              // sentinel slot: hand it back and stop
      __syncwarp();
      if (lane == 0) mbar_arrive(ring.empty0 + 8u * rp.s);
      ring_advance(ring, rp);
      break;
    }
    const int q = plan.unit_entry[lo + u / g.n_chunks], c = u % g.n_chunks;
    const int e = plan.entry_expert[q];
    const int cnt = min(plan.exp_count[e], kDecodeMaxTokens);
    const int pos0 = plan.exp_offset[e];
    const int* pl = plan.pair_list + pos0;
    const bool fill = a.master != nullptr && plan.entry_miss[q] != 0;
    char* slot_blob = const_cast<char*>(a.pool) + ((size_t)plan.entry_slot[q] * a.L + a.layer) * a.blob_bytes;
    int part = 0;
    // hand a consumed ring slot back (after, on a miss, warp 0 has stored it into the victim slot)
    auto store_part = [&](const DecPart& pt) {
      if (fill && warp == 0) {
        if (lane == 0) {
          const int np = pt.mat == 2 ? g.down_pieces : 1;
          const uint32_t pb = (uint32_t)g.part_bytes / np, src = ring.slot0 + (uint32_t)rp.s * ring.stride;
          for (int piece = 0; piece < np; ++piece) bulk_s2g(slot_blob + dec_part_offset(g, c, pt, piece), src + piece * pb, pb);
          bulk_commit();
        }
      }
    };
    auto release = [&]() {
      if (fill && warp == 0 && lane == 0) bulk_wait_read0();   // the bulk store has finished reading the slot
      __syncwarp();
      if (lane == 0) mbar_arrive(ring.empty0 + 8u * rp.s);
      ring_advance(ring, rp);
    };
    const int tok = col < cnt ? pl[col] / a.k : -1;            // token of MMA column `col` (-1: unused column, operand 0)

    // ================= gate/up + SwiGLU, sub-block by sub-block =================
    for (int sb = 0; sb < g.n_sb; ++sb) {
      float cacc[4] = {0.f, 0.f, 0.f, 0.f};                    // MMA: this warp's 16 x 8 partial tile (rows 0-7 gate, 8-15 up)
      for (int s = 0; s < g.n_slab; ++s) {
        // ring slots of the gate part and of the up part
        if (part > 0) mbar_wait(ring.full0 + 8u * rp.s, rp.ph);
        const uint32_t gbase = ring.slot0 + (uint32_t)rp.s * ring.stride;
        const DecPart ptg = dec_part(g, part);
        store_part(ptg);
        DecRingPos rpu = rp;
        ring_advance(ring, rpu);
        mbar_wait(ring.full0 + 8u * rpu.s, rpu.ph);
        const uint32_t ubase = ring.slot0 + (uint32_t)rpu.s * ring.stride;
        const int k_lo = s * g.slab + warp * (g.slab >> 3);    // this warp's K range of the slab
        if constexpr (kMma) {
          const uint32_t abase = ((lane >> 3) & 1 ? ubase : gbase) + (uint32_t)(lane & 7) * 16u + (uint32_t)(lane >> 4) * 128u +
                                 (uint32_t)(warp * g.steps) * 256u;
          const T* xrow = xs + (size_t)max(tok, 0) * xs_pitch + k_lo + kq;
#pragma unroll
          for (int t = 0; t < kDecMaxSteps; ++t) {
            if (t < g.steps) {
              uint32_t a0, a1, a2, a3;
              ldmatrix_x4(a0, a1, a2, a3, abase + (uint32_t)t * 256u);
              uint32_t b0 = 0u, b1 = 0u;
              if (tok >= 0) {
                b0 = *reinterpret_cast<const uint32_t*>(xrow + t * 16);
                b1 = *reinterpret_cast<const uint32_t*>(xrow + t * 16 + 8);
              }
              mma_bf16_16816(cacc, a0, a1, a2, a3, b0, b1);
            }
          }
        } else {
          // fp32: lane l owns the 16-byte chunks l, l+32, ... of the warp's K range; one token column at a time
          const int n_chunk = (g.slab >> 3) / g.kc;
          for (int n = 0; n < cnt; ++n) {
            const T* xrow = xs + (size_t)(pl[n] / a.k) * xs_pitch + k_lo;
            for (int r = 0; r < 16; ++r) {
              const uint32_t base = (r < 8 ? gbase : ubase) + (uint32_t)(r & 7) * 16u + (uint32_t)(warp * n_chunk) * 128u;
              float acc = 0.f;
              for (int ch = lane; ch < n_chunk; ch += 32) {
                float wv[4];
                asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(wv[0]), "=f"(wv[1]), "=f"(wv[2]), "=f"(wv[3]) : "r"(base + (uint32_t)ch * 128u));
#pragma unroll
                for (int j = 0; j < 4; ++j) acc = fmaf(wv[j], to_f32<T>(xrow[ch * 4 + j]), acc);
              }
              acc = warp_sum(acc);
              if (lane == 0) {                                  // accumulates over the slabs of the sub-block
                float* dst = s_red + warp * 128 + cfrag_index(r, n);
                *dst = (s == 0 ? 0.f : *dst) + acc;
              }
            }
          }
        }
        release();                       // gate part
        const DecPart ptu = dec_part(g, part + 1);
        store_part(ptu);
        release();                       // up part
        part += 2;
      }
      // ---- cross-warp reduction (ascending warp order) + SwiGLU, by warp 0 ----
      if constexpr (kMma) {
        *reinterpret_cast<float4*>(s_red + warp * 128 + lane * 4) = make_float4(cacc[0], cacc[1], cacc[2], cacc[3]);
      }
      asm volatile("bar.sync 1, 256;" ::: "memory");
      if (warp == 0) {
        float4 tot = *reinterpret_cast<const float4*>(s_red + lane * 4);
#pragma unroll
        for (int w = 1; w < kDecWarps; ++w) {
          const float4 v = *reinterpret_cast<const float4*>(s_red + w * 128 + lane * 4);
          tot.x += v.x; tot.y += v.y; tot.z += v.z; tot.w += v.w;
        }
        // lane holds gate (x, y) and up (z, w) of act row lane/4 for token columns kq, kq+1
        AT* dst = s_act + (sb * 8) * 8;
        if constexpr (kMma) {
          dst[(kq) * 8 + col] = __float2bfloat16_rn(silu_f(tot.x) * tot.z);
          dst[(kq + 1) * 8 + col] = __float2bfloat16_rn(silu_f(tot.y) * tot.w);
        } else {
          dst[(kq) * 8 + col] = silu_f(tot.x) * tot.z;
          dst[(kq + 1) * 8 + col] = silu_f(tot.y) * tot.w;
        }
      }
      asm volatile("bar.sync 1, 256;" ::: "memory");
    }

    // ================= down: P[pair][c][j] = sum_i a_i * D[j][i], slab by slab =================
    for (int s = 0; s < g.n_slab; ++s) {
      float yacc[kMma ? kDecMaxSteps : 1][4];
      if constexpr (kMma) {
#pragma unroll
        for (int t = 0; t < kDecMaxSteps; ++t) { yacc[t][0] = 0.f; yacc[t][1] = 0.f; yacc[t][2] = 0.f; yacc[t][3] = 0.f; }
      }
      for (int sb = 0; sb < g.n_sb; ++sb) {
        mbar_wait(ring.full0 + 8u * rp.s, rp.ph);
        const uint32_t dbase = ring.slot0 + (uint32_t)rp.s * ring.stride;
        const DecPart ptd = dec_part(g, part);
        store_part(ptd);
        if constexpr (kMma) {
          // A[j][i]: 16 outputs j x (8 act columns i, upper half of K zero); B[i][n] = a[n][i]
          const uint32_t b0 = *reinterpret_cast<const uint32_t*>(s_act + (sb * 8 + col) * 8 + kq);
          const uint32_t abase = dbase + (uint32_t)(lane & 7) * 16u + (uint32_t)((lane >> 3) & 1) * 128u + (uint32_t)(warp * g.steps) * 256u;
#pragma unroll
          for (int t = 0; t < kDecMaxSteps; ++t) {
            if (t < g.steps) {
              uint32_t a0, a1;
              ldmatrix_x2(a0, a1, abase + (uint32_t)t * 256u);
              mma_bf16_16816(yacc[t], a0, a1, 0u, 0u, b0, 0u);
            }
          }
        } else {
          // fp32: thread owns outputs j = tid, tid + 256, ... of the slab; n_sb == 1 for fp32 models, so the sum over the 8 act
          // columns is complete here: i ascending, fmaf from 0.f
          const uint32_t half = (uint32_t)g.part_bytes / 2;
          for (int jj = tid; jj < g.slab; jj += kDecConsumers) {
            float wv[8];
            const uint32_t addr = dbase + (uint32_t)(jj >> 3) * 128u + (uint32_t)(jj & 7) * 16u;
            asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(wv[0]), "=f"(wv[1]), "=f"(wv[2]), "=f"(wv[3]) : "r"(addr));
            asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(wv[4]), "=f"(wv[5]), "=f"(wv[6]), "=f"(wv[7]) : "r"(addr + half));
            for (int n = 0; n < cnt; ++n) {
              float acc = 0.f;
#pragma unroll
              for (int i = 0; i < 8; ++i) acc = fmaf(wv[i], to_f32<AT>(s_act[(sb * 8 + n) * 8 + i]), acc);
              a.partial[((size_t)(pos0 + n) * g.n_chunks + c) * g.d + s * g.slab + jj] = acc;
            }
          }
        }
        release();
        ++part;
      }
      if constexpr (kMma) {
        const int j0 = s * g.slab + warp * (g.slab >> 3) + col;
        float* p0 = a.partial + ((size_t)(pos0 + kq) * g.n_chunks + c) * g.d + j0;
        float* p1 = p0 + (size_t)g.n_chunks * g.d;
#pragma unroll
        for (int t = 0; t < kDecMaxSteps; ++t) {
          if (t < g.steps) {
            if (kq < cnt) { p0[t * 16] = yacc[t][0]; p0[t * 16 + 8] = yacc[t][2]; }
            if (kq + 1 < cnt) { p1[t * 16] = yacc[t][1]; p1[t * 16 + 8] = yacc[t][3]; }
          }
        }
      }
    }
  }
  if (a.master != nullptr && tid == 0) bulk_wait0();     // this CTA's slot fills are complete before the next grid-wide barrier
}

}  // namespace wisp
