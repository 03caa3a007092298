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
// Data path per CTA (320 threads), a dataflow of four roles that talk through mbarriers only (no block-wide barrier):
//   producer warp (one lane): takes unit tickets and streams each unit's parts (8 rows x one slab of at most 32 KiB) through
//     a shared-memory ring with 1-D TMA bulk copies (cp.async.bulk + mbarrier complete_tx), in the order
//     gate/up(unit i+1), down(unit i), ... so the down parts of a unit arrive while its SwiGLU is being reduced;
//   8 consumer warps: gate/up of a sub-block of 8 act rows -- warp w owns the K range [w, w+1) * slab/8 of every slab and
//     leaves its 16 x 8 partial tile (rows 0-7 gate, 8-15 up; columns = the tokens routed to the expert) in shared memory;
//     down -- warp w owns the outputs j in [w, w+1) * slab/8 of every slab, accumulates over the chunk's rows in registers
//     and stores the chunk partial.  Each warp runs at its own pace; a ring slot is free when all 8 warps have read it;
//   reducer warp: adds the 8 warps' gate/up partials in ascending warp order, applies SwiGLU, publishes
//     a[8 rows][8 tokens] (bf16 for bf16 models, G21) for the down parts.
// bf16: the products run on the tensor cores through mma.sync.m16n8k16 (A fragments come straight from the ring with
// ldmatrix, each core matrix being 128 contiguous bytes), so the arithmetic leaves the FMA pipes and the kernel stays a pure
// HBM stream at 1..8 tokens (1 flop/byte: this is an ALU offload of a memory-bound kernel, not a GEMM -- units of 96 KiB are
// far too small for tcgen05's 128-row tiles).  fp32 (config 1, parity only): plain FMA, same data flow, same reduction tree.
// fp8 experts (WISP_FP8_E4M3, f4): the slot holds e4m3 codes in the same 8-row x 16-byte cores (16 K elements per row
// of a gate/up core; down cores are 8 outputs x 8 act columns = 64 bytes) and the fp32 block scales at the blob's tail; every
// part carries its slab/128 scales behind its data in the ring slot.  ldmatrix delivers 4 consecutive K codes per lane; since
// the order of k inside one MMA is free as long as A and B agree, they feed the k slots {2q, 2q+1, 2q+8, 2q+9} of lane
// quarter q directly -- no shuffles: two exact cvt.f16x2.e4m3x2 per register, the activations (hidden state, a) as f16 scaled
// by an exact per-token power of two, f16 MMA with fp32 accumulation, one 128-wide K block per accumulator, block sums
// scaled in fp32 (fmaf) in ascending block order.  Every product is exact; only the fp32 accumulation rounds.
// Fused miss path (WISP_FETCH_FUSED): the parts of an entry marked as a miss are read from the mapped pinned master
// (Alg. 1 line 6) and consumer warp 0 stores each landed part into the victim slot with a bulk shared->global
// copy: same bytes, same order of arithmetic as a hit.
#pragma once
#include "common.cuh"

namespace wisp {

constexpr int kDecConsumers = 256;                      // 8 consumer warps
constexpr int kDecWarps = kDecConsumers / 32;
constexpr int kDecThreads = kDecConsumers + 64;         // + producer warp + reducer warp
constexpr int kDecMaxSlots = 8;
constexpr int kDecMaxSteps = 16;                        // MMA steps per warp per part: slab / 128 <= 16
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
  // fp8 experts: fp32 block scales at the tail of the blob, S13 [2 d_ff / 128][d / 128] then S2 TRANSPOSED [d_ff / 128][d / 128]
  int f8;                // 1: e4m3 weights with block scales
  int act_elem;          // bytes per hidden-state element (2 for fp8 experts)
  int scale_bytes;       // per part: 4 * slab / 128 (0 without scales)
  int slot_bytes;        // ring slot = part_bytes + scale_bytes
  int merge;             // 1: one part holds ALL sub-blocks of the unit (consecutive 8-row groups are contiguous; fp8 with n_slab == 1):
                         //    the producer lane's cost per part is what bounds 16 KiB parts, so fp8 parts are 32 KiB like bf16's
  int sub_bytes;         // 8 * slab * elem: one sub-block inside a part
  unsigned long long s13_off, s2_off;
};

struct DecodeFfnArgs {
  const char* layer_base; // slot s of this layer at layer_base + s * slot_stride.  Paged pool: arena + layer * M_e with stride L * M_e
  unsigned long long slot_stride;   //   (slot-major arena); static-offload arm: the layer's own region with stride M_e
  const char* master;     // mapped pinned master of this layer (fused miss path) or nullptr
  unsigned long long blob_bytes;
  int k;
  float inv_k;            // 1.0f / k (token of pair p = floor((p + 0.5) / k), exact for p < 256)
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

// One ring part: matrix (0 gate, 1 up, 2 down), sub-block of 8 act rows inside the unit, slab of d.
struct DecPart { int mat, sb, slab; };
// What the producer tells the consumers about the part in a ring slot (one int per slot).
constexpr int kPartEnd = 3;
__device__ __forceinline__ int part_meta(int kind, int sb, int slab, int c, int q) { return kind | (sb << 2) | (slab << 4) | (c << 8) | (q << 20); }
// Byte offset inside the blob of piece `piece` of that part.
__device__ __forceinline__ unsigned long long dec_part_offset(const DecodeGeom& g, int c, const DecPart& p, int piece) {
  const unsigned long long grp = (unsigned long long)(c * g.n_sb + p.sb);
  if (p.mat < 2) return (p.mat ? g.up_off : 0ull) + grp * g.group_bytes + (unsigned long long)p.slab * g.part_bytes;
  const unsigned long long pb = (unsigned long long)g.part_bytes / g.down_pieces;
  return g.down_off + (grp * g.down_pieces + piece) * (g.group_bytes / g.down_pieces) + (unsigned long long)p.slab * pb;
}

// Byte offset inside the blob of the block scales of that part (fp8): the slab/128 scales of its K range (gate/up: row block of the
// 8 rows) or of its output range (down: column block of the 8 act columns; S2 is stored transposed so they are contiguous).
__device__ __forceinline__ unsigned long long dec_scale_offset(const DecodeGeom& g, int c, const DecPart& p) {
  const int row0 = (c * g.n_sb + p.sb) * 8;
  const unsigned long long blk = p.mat < 2 ? (unsigned long long)((p.mat * g.dff + row0) >> 7) : (unsigned long long)(row0 >> 7);
  return (p.mat < 2 ? g.s13_off : g.s2_off) + 4ull * (blk * (unsigned long long)(g.d >> 7)) + (unsigned long long)p.slab * g.scale_bytes;
}

// ---- per-CTA dataflow state (shared memory) -----------------------------------------------------------------------
struct DecFfnShared {
  unsigned long long full[kDecMaxSlots], empty[kDecMaxSlots];
  unsigned long long red_full[2][2];     // [unit parity][sub-block]: the 8 consumer warps' gate/up partials are in place
  unsigned long long act_ready[2];       // [unit parity]: the reducer has published a[] of every sub-block of the unit
  int meta[kDecMaxSlots];                // part_meta of the part in each ring slot
  volatile int units_total;              // units this CTA's producer has queued so far (all waves of the launch)
  volatile int final;                    // the consumers have finished the last wave of the launch
  int abort;                             // a grid barrier timed out: everybody leaves
  alignas(16) float red[2][2][kDecWarps * 128];   // gate/up partial tiles; also the combine's scratch between waves
  alignas(16) float act[2][2][64];       // a[token column][act row] per (unit parity, sub-block), bf16 or fp32 (fp8 experts: scaled f16)
  // fp8 experts: exact power-of-two scales of the f16 activation operands
  float xscale[kDecodeMaxTokens];        // hidden state of token t = xh[t] * xscale[t]
  unsigned xamax[kDecodeMaxTokens];      // scratch of stage_xh
  float colscale[2][8];                  // [unit parity][MMA column]: xscale of the column's token (written by consumer warp 0)
  float ascale[2][8];                    // [unit parity][MMA column]: a = act * ascale (written by the reducer)
};

__device__ __forceinline__ void dec_ffn_shared_init(DecFfnShared& fs, const DecRing& ring) {   // one thread, before a CTA-wide sync
  ring_init(ring);
  for (int p = 0; p < 2; ++p) {
    mbar_init(smem_u32(&fs.act_ready[p]), 1);
    for (int sb = 0; sb < 2; ++sb) mbar_init(smem_u32(&fs.red_full[p][sb]), kDecWarps);
  }
  mbar_fence_init();
  fs.units_total = 0; fs.final = 0; fs.abort = 0;
}

// Exact power-of-two factor that brings a non-negative fp32 maximum into [2^14, 2^15) (f16 range), and its inverse.
__device__ __forceinline__ void f16_range_scale(float amax, float& mult, float& inv) {
  const unsigned e = max(15u, (__float_as_uint(amax) >> 23) & 0xffu);
  mult = __uint_as_float((268u - e) << 23);
  inv = __uint_as_float((e - 14u) << 23);
}

// fp8 experts: the f16 copy of the call's hidden states, xh[t] = xs[t] * 2^p_t with the token's largest magnitude brought into
// [2^14, 2^15) (exact: bf16 has fewer mantissa bits than f16; elements more than 2^29 below the token's maximum round to f16
// subnormals, an absolute error below 2^-39 of that maximum).  Called by `nthreads` threads that `bar()` synchronises; xs must be
// complete before the call, and the caller synchronises once more before xh / xscale are read.
template <typename Bar>
__device__ __forceinline__ void stage_xh(const __nv_bfloat16* xs, __half* xh, DecFfnShared& fs, int n_tokens, int d, int pitch, int tid,
                                         int nthreads, Bar bar) {
  if (tid < kDecodeMaxTokens) fs.xamax[tid] = 0u;
  bar();
  const int vec_row = d / 8, n_vec = n_tokens * vec_row;        // a warp's 32 consecutive vectors lie in one token (d % 256 == 0)
  for (int i0 = 0; i0 < n_vec; i0 += nthreads) {
    const int i = i0 + tid;
    unsigned m = 0u;
    if (i < n_vec) {
      const uint4 v = *reinterpret_cast<const uint4*>(xs + (size_t)(i / vec_row) * pitch + (i % vec_row) * 8);
      const unsigned w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
      for (int j = 0; j < 4; ++j) m = max(m, max(w[j] & 0x7fffu, (w[j] >> 16) & 0x7fffu));
    }
    m = __reduce_max_sync(0xffffffffu, m);
    if ((tid & 31) == 0 && i < n_vec) atomicMax(&fs.xamax[i / vec_row], m);
  }
  bar();
  for (int i = tid; i < n_vec; i += nthreads) {
    const int t = i / vec_row;
    float mult, inv;
    f16_range_scale(__uint_as_float(fs.xamax[t] << 16), mult, inv);
    if (i % vec_row == 0) fs.xscale[t] = inv;
    const size_t off = (size_t)t * pitch + (i % vec_row) * 8;
    const uint4 v = *reinterpret_cast<const uint4*>(xs + off);
    const unsigned w[4] = {v.x, v.y, v.z, v.w};
    unsigned o[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const __half2 h = __floats2half2_rn(__uint_as_float(w[j] << 16) * mult, __uint_as_float(w[j] & 0xffff0000u) * mult);
      o[j] = *reinterpret_cast<const unsigned*>(&h);
    }
    *reinterpret_cast<uint4*>(xh + off) = make_uint4(o[0], o[1], o[2], o[3]);
  }
}

__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
  uint32_t done;
  asm volatile("{\n.reg .pred P1;\nmbarrier.try_wait.parity.shared::cta.b64 P1, [%1], %2;\nselp.u32 %0, 1, 0, P1;\n}"
               : "=r"(done) : "r"(bar), "r"(parity) : "memory");
  return done != 0;
}
// mbarrier wait that gives up when the CTA aborted (a grid barrier timed out)
__device__ __forceinline__ bool mbar_wait_or_abort(uint32_t bar, uint32_t parity, const int* s_abort) {
  while (!mbar_try_wait(bar, parity))
    if (*reinterpret_cast<const volatile int*>(s_abort)) return false;
  return true;
}

// ---- producer: one lane takes unit tickets and issues the bulk loads --------------------------------------------
// Units of the wave whose plan entries are [lo, lo + nw): u in [0, nw * NC), entry = unit_entry[lo + u / NC], chunk = u % NC.
// The first unit of CTA b is b (no atomic on the critical path of a phase start), later ones come from the ticket counter.
// Part order in the ring: gate/up parts of unit i+1 (sub-block major, slab minor, gate before up), then the down parts of
// unit i (slab major, sub-block minor), ..., the down parts of the last unit, an END marker.
template <bool F8>
__device__ __forceinline__ void decode_produce(const DecodeFfnArgs& a, const DecodeGeom& g, const PlanPtrs& plan, DecFfnShared& fs,
                                               const DecRing& ring, DecRingPos& rp, int lo, int nw, uint64_t pol) {
  const int n_units = nw * g.n_chunks;
  auto emit = [&](const char* blob, int q, int c, const DecPart& pt) -> bool {
    if (!mbar_wait_or_abort(ring.empty0 + 8u * rp.s, rp.ph ^ 1u, &fs.abort)) return false;
    fs.meta[rp.s] = part_meta(pt.mat, pt.sb, pt.slab, c, q);
    const uint32_t bar = ring.full0 + 8u * rp.s, dst = ring.slot0 + (uint32_t)rp.s * ring.stride;
    mbar_expect_tx(bar, F8 ? (uint32_t)g.slot_bytes : (uint32_t)g.part_bytes);
    const int np = pt.mat == 2 ? g.down_pieces : 1;
    const uint32_t pb = (uint32_t)g.part_bytes / np;
    for (int piece = 0; piece < np; ++piece) bulk_g2s(dst + piece * pb, blob + dec_part_offset(g, c, pt, piece), pb, bar, pol);
    if constexpr (F8) bulk_g2s(dst + (uint32_t)g.part_bytes, blob + dec_scale_offset(g, c, pt), (uint32_t)g.scale_bytes, bar, pol);
    ring_advance(ring, rp);
    return true;
  };
  auto blob_of = [&](int q) {
    const bool from_host = a.master != nullptr && plan.entry_miss[q] != 0;
    return from_host ? a.master + (size_t)plan.entry_expert[q] * a.blob_bytes
                     : a.layer_base + (size_t)plan.entry_slot[q] * a.slot_stride;
  };
  auto emit_down = [&](int q, int c) -> bool {
    const char* blob = blob_of(q);
    for (int s = 0; s < g.n_slab; ++s)
      for (int sb = 0; sb < (F8 && g.merge ? 1 : g.n_sb); ++sb)
        if (!emit(blob, q, c, DecPart{2, sb, s})) return false;
    return true;
  };
  int u = (int)blockIdx.x, pq = -1, pc = 0, count = 0;
  while (u < n_units) {
    const unsigned t = atomicAdd(a.ticket, 1u);                // next unit: its latency hides behind this unit's copies
    const int q = plan.unit_entry[lo + u / g.n_chunks], c = u % g.n_chunks;
    const char* blob = blob_of(q);
    for (int sb = 0; sb < (F8 && g.merge ? 1 : g.n_sb); ++sb)
      for (int s = 0; s < g.n_slab; ++s) {
        if (!emit(blob, q, c, DecPart{0, sb, s})) return;
        if (!emit(blob, q, c, DecPart{1, sb, s})) return;
      }
    if (pq >= 0 && !emit_down(pq, pc)) return;
    pq = q; pc = c; ++count;
    u = (int)gridDim.x + (int)t;
  }
  if (pq >= 0 && !emit_down(pq, pc)) return;
  if (!mbar_wait_or_abort(ring.empty0 + 8u * rp.s, rp.ph ^ 1u, &fs.abort)) return;   // END marker: this wave is over
  fs.meta[rp.s] = kPartEnd;
  mbar_arrive(ring.full0 + 8u * rp.s);
  ring_advance(ring, rp);
  fs.units_total = fs.units_total + count;
}

// C-fragment position of element (row, col) of a 16 x 8 tile inside a warp's 128-float partial (index lane * 4 + reg).
__device__ __forceinline__ int cfrag_index(int row, int col) { return ((row & 7) * 4 + (col >> 1)) * 4 + ((row >> 3) << 1) + (col & 1); }

template <typename T> struct ActT { typedef float type; };
template <> struct ActT<__nv_bfloat16> { typedef __nv_bfloat16 type; };

// ---- reducer warp: SwiGLU of every unit the consumers push, until the launch is over ------------------------------
// a[n][r] = silu(sum_w gate_w[r][n]) * (sum_w up_w[r][n]), the 8 warp partials added in ascending warp order.
template <typename T, bool F8>
__device__ __forceinline__ void decode_reduce(const DecodeGeom& g, DecFfnShared& fs, int lane) {
  typedef typename ActT<T>::type AT;
  const int col = lane >> 2, kq = (lane & 3) * 2;
  for (unsigned i = 0;; ++i) {
    const unsigned par = i & 1u, ph = (i >> 1) & 1u;
    float av[2][2];                                            // fp8: a of (sub-block, column kq / kq+1) until the unit's scale is known
    for (int sb = 0; sb < g.n_sb; ++sb) {
      const uint32_t bar = smem_u32(&fs.red_full[par][sb]);
      while (!mbar_try_wait(bar, ph))
        if (fs.abort || (fs.final && (int)i >= fs.units_total)) return;
      const float* red = fs.red[par][sb];
      float4 tot = *reinterpret_cast<const float4*>(red + lane * 4);
#pragma unroll
      for (int w = 1; w < kDecWarps; ++w) {
        const float4 v = *reinterpret_cast<const float4*>(red + w * 128 + lane * 4);
        tot.x += v.x; tot.y += v.y; tot.z += v.z; tot.w += v.w;
      }
      // this lane holds gate (x, y) and up (z, w) of act row lane/4 for the token columns kq, kq+1
      AT* dst = reinterpret_cast<AT*>(fs.act[par][sb]);
      if constexpr (F8) {
        // the operands were xh = x / xscale: put the token's power of two back (exact), then a in the model's bf16 (G21)
        const float c0 = fs.colscale[par][kq], c1 = fs.colscale[par][kq + 1];
        av[sb & 1][0] = __bfloat162float(__float2bfloat16_rn(silu_f(tot.x * c0) * (tot.z * c0)));
        av[sb & 1][1] = __bfloat162float(__float2bfloat16_rn(silu_f(tot.y * c1) * (tot.w * c1)));
      } else if constexpr (sizeof(T) == 2) {
        dst[kq * 8 + col] = __float2bfloat16_rn(silu_f(tot.x) * tot.z);
        dst[(kq + 1) * 8 + col] = __float2bfloat16_rn(silu_f(tot.y) * tot.w);
      } else {
        dst[kq * 8 + col] = silu_f(tot.x) * tot.z;
        dst[(kq + 1) * 8 + col] = silu_f(tot.y) * tot.w;
      }
    }
    if constexpr (F8) {
      // one scale per (unit, token column): the column's largest |a| over the unit's rows -> [2^14, 2^15); a is bf16, so the scaled
      // f16 operand is exact
      float m0 = fabsf(av[0][0]), m1 = fabsf(av[0][1]);
      if (g.n_sb > 1) { m0 = fmaxf(m0, fabsf(av[1][0])); m1 = fmaxf(m1, fabsf(av[1][1])); }
#pragma unroll
      for (int o = 4; o < 32; o <<= 1) {
        m0 = fmaxf(m0, __shfl_xor_sync(0xffffffffu, m0, o));
        m1 = fmaxf(m1, __shfl_xor_sync(0xffffffffu, m1, o));
      }
      float mu0, in0, mu1, in1;
      f16_range_scale(m0, mu0, in0);
      f16_range_scale(m1, mu1, in1);
      for (int sb = 0; sb < g.n_sb; ++sb) {
        __half* dst = reinterpret_cast<__half*>(fs.act[par][sb]);
        dst[kq * 8 + col] = __float2half_rn(av[sb & 1][0] * mu0);
        dst[(kq + 1) * 8 + col] = __float2half_rn(av[sb & 1][1] * mu1);
      }
      if (col == 0) { fs.ascale[par][kq] = in0; fs.ascale[par][kq + 1] = in1; }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(smem_u32(&fs.act_ready[par]));
  }
}

// ---- consumers: the 8 warps (tid 0..255) process the parts the producer queued, until the END marker ---------------
// xs: the call's hidden states in shared memory, [T][xs_pitch] elements of T (rows padded by 16 bytes).
// gu_seq / d_seq: units whose gate/up / down this warp has finished so far in the launch (select the parity buffers).
// fp8 experts: xh = the hidden states as f16 scaled per token (stage_xh), same pitch as xs.
template <typename T, bool F8>
__device__ __forceinline__ void decode_consume(const DecodeFfnArgs& a, const DecodeGeom& g, const PlanPtrs& plan, DecFfnShared& fs,
                                               const DecRing& ring, DecRingPos& rp, unsigned& gu_seq, unsigned& d_seq, const T* xs,
                                               const __half* xh, int xs_pitch) {
  typedef typename ActT<T>::type AT;
  constexpr bool kMma = sizeof(T) == 2 && !F8;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int col = lane >> 2, kq = (lane & 3) * 2;             // MMA fragment coordinates of this lane
  while (true) {
    mbar_wait(ring.full0 + 8u * rp.s, rp.ph);
    const int meta = fs.meta[rp.s];
    const int kind = meta & 3;
    if (kind == kPartEnd) {                                   // hand the marker's slot back and stop
      __syncwarp();
      if (lane == 0) mbar_arrive(ring.empty0 + 8u * rp.s);
      ring_advance(ring, rp);
      break;
    }
    // The part opens a GROUP of parts of the same unit: kind 0 = the gate/up parts of sub-block sb0 (n_slab pairs), kind 2 =
    // the down parts of slab s0 (n_sb parts).  The accumulators of a group live only inside it.
    const int sb0 = (meta >> 2) & 3, s0 = (meta >> 4) & 15, c = (meta >> 8) & 0xfff, q = (meta >> 20) & 0x3ff;
    const int e = plan.entry_expert[q];
    const int cnt = min(plan.exp_count[e], kDecodeMaxTokens);
    const int pos0 = plan.exp_offset[e];
    const int* pl = plan.pair_list + pos0;
    const bool fill = a.master != nullptr && plan.entry_miss[q] != 0;
    char* slot_blob = const_cast<char*>(a.layer_base) + (size_t)plan.entry_slot[q] * a.slot_stride;
    // on a miss, warp 0 stores the landed part into the victim slot before the ring slot is handed back
    auto store_part = [&](const DecPart& pt, int ring_slot = -1) {
      if (fill && warp == 0 && lane == 0) {
        const int np = pt.mat == 2 ? g.down_pieces : 1;
        const uint32_t pb = (uint32_t)g.part_bytes / np, src = ring.slot0 + (uint32_t)(ring_slot < 0 ? rp.s : ring_slot) * ring.stride;
        for (int piece = 0; piece < np; ++piece) bulk_s2g(slot_blob + dec_part_offset(g, c, pt, piece), src + piece * pb, pb);
        if constexpr (F8) bulk_s2g(slot_blob + dec_scale_offset(g, c, pt), src + (uint32_t)g.part_bytes, (uint32_t)g.scale_bytes);
        bulk_commit();
      }
    };
    auto release = [&]() {
      if (fill && warp == 0 && lane == 0) bulk_wait_read0();   // the bulk store has finished reading the slot
      __syncwarp();
      if (lane == 0) mbar_arrive(ring.empty0 + 8u * rp.s);
      ring_advance(ring, rp);
    };

    if (kind == 0) {
      // ================= gate/up group of sub-block sb (each gate part is followed by its up part) =================
      // the warp's 16 x 8 partial tile (rows 0-7 gate, 8-15 up) as FOUR independent accumulator chains (k-step t feeds chain
      // t % 4), added as (0 + 1) + (2 + 3) when the last slab is done
      const int sb = sb0;
      float c4[4][4];
#pragma unroll
      for (int j = 0; j < 4; ++j) { c4[j][0] = 0.f; c4[j][1] = 0.f; c4[j][2] = 0.f; c4[j][3] = 0.f; }
      float tot8[4] = {0.f, 0.f, 0.f, 0.f};                    // fp8: the scaled block sums of this warp's K ranges, slabs ascending
      const unsigned par = gu_seq & 1u;
      float* red = fs.red[par][sb] + warp * 128;
      if constexpr (F8) {
        // the reducer needs each MMA column's token scale: warp 0 publishes them with the first sub-block
        if (sb == 0 && warp == 0 && lane < 8)
          fs.colscale[par][lane] = lane < cnt ? fs.xscale[(int)(((float)pl[lane] + 0.5f) * a.inv_k)] : 0.f;
      }
      for (int s = 0; s < g.n_slab; ++s) {
      if (s > 0) mbar_wait(ring.full0 + 8u * rp.s, rp.ph);
      const uint32_t gbase = ring.slot0 + (uint32_t)rp.s * ring.stride;
      store_part(DecPart{0, sb, s});
      DecRingPos rpu = rp;
      ring_advance(ring, rpu);
      mbar_wait(ring.full0 + 8u * rpu.s, rpu.ph);
      const uint32_t ubase = ring.slot0 + (uint32_t)rpu.s * ring.stride;
      const int k_lo = s * g.slab + warp * (g.slab >> 3);     // this warp's K range of the slab
      if constexpr (F8) {
        // one core matrix (8 rows x 16 codes) is one k16 step; an ldmatrix.x4 = {gate, up} x two steps; 8 steps = one scale block.
        // A merged part (g.merge) holds every sub-block of the unit: they are computed one after the other from the same two slots.
        const int tok = col < cnt ? (int)(((float)pl[col] + 0.5f) * a.inv_k) : -1;
        const __half* xrow = xh + (size_t)max(tok, 0) * xs_pitch + k_lo + (lane & 3) * 4;
        const uint32_t sc = (uint32_t)g.part_bytes + (uint32_t)(warp * (g.steps >> 3)) * 4u;
        const int n_in = g.merge ? g.n_sb : 1;
        for (int sbi = 0; sbi < n_in; ++sbi) {
          const uint32_t abase = ((lane >> 3) & 1 ? ubase : gbase) + (uint32_t)sbi * (uint32_t)g.sub_bytes + (uint32_t)(lane & 7) * 16u +
                                 (uint32_t)(lane >> 4) * 128u + (uint32_t)(warp * g.steps) * 128u;
          if (g.merge) { tot8[0] = 0.f; tot8[1] = 0.f; tot8[2] = 0.f; tot8[3] = 0.f; }
#pragma unroll
          for (int kb = 0; kb < kDecMaxSteps / 8; ++kb) {
            if (kb * 8 < g.steps) {
              uint32_t af[4][4];
              uint2 bf[8];
#pragma unroll
              for (int j = 0; j < 4; ++j) {
                ldmatrix_x4(af[j][0], af[j][1], af[j][2], af[j][3], abase + (uint32_t)(kb * 4 + j) * 256u);
                bf[2 * j] = tok >= 0 ? *reinterpret_cast<const uint2*>(xrow + (kb * 8 + 2 * j) * 16) : make_uint2(0u, 0u);
                bf[2 * j + 1] = tok >= 0 ? *reinterpret_cast<const uint2*>(xrow + (kb * 8 + 2 * j + 1) * 16) : make_uint2(0u, 0u);
              }
              float c8[4][4];
#pragma unroll
              for (int j = 0; j < 4; ++j) {
                // registers 0/1: gate / up codes of step 2j; registers 2/3: of step 2j + 1.  Chain (2j) & 3 / (2j + 1) & 3; the first
                // product of a chain starts from a zero accumulator
                const uint32_t g0 = cvt_e4m3x2_f16x2((uint16_t)af[j][0]), u0 = cvt_e4m3x2_f16x2((uint16_t)af[j][1]);
                const uint32_t g1 = cvt_e4m3x2_f16x2((uint16_t)(af[j][0] >> 16)), u1 = cvt_e4m3x2_f16x2((uint16_t)(af[j][1] >> 16));
                const uint32_t g2 = cvt_e4m3x2_f16x2((uint16_t)af[j][2]), u2 = cvt_e4m3x2_f16x2((uint16_t)af[j][3]);
                const uint32_t g3 = cvt_e4m3x2_f16x2((uint16_t)(af[j][2] >> 16)), u3 = cvt_e4m3x2_f16x2((uint16_t)(af[j][3] >> 16));
                if (j < 2) {
                  mma_f16_16816_zero(c8[(2 * j) & 3], g0, u0, g1, u1, bf[2 * j].x, bf[2 * j].y);
                  mma_f16_16816_zero(c8[(2 * j + 1) & 3], g2, u2, g3, u3, bf[2 * j + 1].x, bf[2 * j + 1].y);
                } else {
                  mma_f16_16816(c8[(2 * j) & 3], g0, u0, g1, u1, bf[2 * j].x, bf[2 * j].y);
                  mma_f16_16816(c8[(2 * j + 1) & 3], g2, u2, g3, u3, bf[2 * j + 1].x, bf[2 * j + 1].y);
                }
              }
              const float sg = lds_f32(gbase + sc + (uint32_t)kb * 4u), su = lds_f32(ubase + sc + (uint32_t)kb * 4u);
              tot8[0] = fmaf(sg, (c8[0][0] + c8[1][0]) + (c8[2][0] + c8[3][0]), tot8[0]);
              tot8[1] = fmaf(sg, (c8[0][1] + c8[1][1]) + (c8[2][1] + c8[3][1]), tot8[1]);
              tot8[2] = fmaf(su, (c8[0][2] + c8[1][2]) + (c8[2][2] + c8[3][2]), tot8[2]);
              tot8[3] = fmaf(su, (c8[0][3] + c8[1][3]) + (c8[2][3] + c8[3][3]), tot8[3]);
            }
          }
          if (g.merge) {                                         // (n_slab == 1) sub-block sbi is complete: hand its tile to the reducer
            *reinterpret_cast<float4*>(fs.red[par][sbi] + warp * 128 + lane * 4) = make_float4(tot8[0], tot8[1], tot8[2], tot8[3]);
            __syncwarp();
            if (lane == 0) mbar_arrive(smem_u32(&fs.red_full[par][sbi]));
          }
        }
        if (!g.merge && s == g.n_slab - 1) *reinterpret_cast<float4*>(red + lane * 4) = make_float4(tot8[0], tot8[1], tot8[2], tot8[3]);
      } else if constexpr (kMma) {
        const int tok = col < cnt ? (int)(((float)pl[col] + 0.5f) * a.inv_k) : -1;   // token of MMA column `col` (-1: operand 0)
        const uint32_t abase = ((lane >> 3) & 1 ? ubase : gbase) + (uint32_t)(lane & 7) * 16u + (uint32_t)(lane >> 4) * 128u +
                               (uint32_t)(warp * g.steps) * 256u;
        const T* xrow = xs + (size_t)max(tok, 0) * xs_pitch + k_lo + kq;
#pragma unroll
        for (int t0 = 0; t0 < kDecMaxSteps; t0 += 4) {
          if (t0 < g.steps) {
            uint32_t af[4][4], bf[4][2];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
              if (t0 + j < g.steps) {
                ldmatrix_x4(af[j][0], af[j][1], af[j][2], af[j][3], abase + (uint32_t)(t0 + j) * 256u);
                bf[j][0] = tok >= 0 ? *reinterpret_cast<const uint32_t*>(xrow + (t0 + j) * 16) : 0u;
                bf[j][1] = tok >= 0 ? *reinterpret_cast<const uint32_t*>(xrow + (t0 + j) * 16 + 8) : 0u;
              }
            }
#pragma unroll
            for (int j = 0; j < 4; ++j)
              if (t0 + j < g.steps) mma_bf16_16816(c4[j], af[j][0], af[j][1], af[j][2], af[j][3], bf[j][0], bf[j][1]);
          }
        }
        if (s == g.n_slab - 1)
          *reinterpret_cast<float4*>(red + lane * 4) =
              make_float4((c4[0][0] + c4[1][0]) + (c4[2][0] + c4[3][0]), (c4[0][1] + c4[1][1]) + (c4[2][1] + c4[3][1]),
                          (c4[0][2] + c4[1][2]) + (c4[2][2] + c4[3][2]), (c4[0][3] + c4[1][3]) + (c4[2][3] + c4[3][3]));
      } else {
        // fp32: lane l owns the 16-byte chunks l, l+32, ... of the warp's K range; one token column at a time; the warp's tile
        // entry accumulates over the slabs in shared memory (warp-private)
        const int n_chunk = (g.slab >> 3) / g.kc;
        for (int n = 0; n < cnt; ++n) {
          const T* xrow = xs + (size_t)(int)(((float)pl[n] + 0.5f) * a.inv_k) * xs_pitch + k_lo;
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
            if (lane == 0) {
              float* dst = red + cfrag_index(r, n);
              *dst = (s == 0 ? 0.f : *dst) + acc;
            }
          }
        }
      }
      release();                                               // gate part
      store_part(DecPart{1, sb, s});
      release();                                               // up part
      }
      if (!(F8 && g.merge)) {
        __syncwarp();                                          // the sub-block's partial tile is complete: tell the reducer
        if (lane == 0) mbar_arrive(smem_u32(&fs.red_full[par][sb]));
      }
      if (sb == g.n_sb - 1 || (F8 && g.merge)) ++gu_seq;
    } else {
      // ================= down group of slab s: P[pair][c][j] = sum_{i in chunk} a_i * D[j][i] for the outputs j of the slab =================
      const int s = s0;
      const unsigned par = d_seq & 1u;
      if (s == 0) mbar_wait(smem_u32(&fs.act_ready[par]), (d_seq >> 1) & 1u);   // a[] of this unit is published
      float yacc[(kMma || F8) ? kDecMaxSteps : 1][4];          // outputs j of this warp x token columns
      if constexpr (kMma || F8) {
#pragma unroll
        for (int t = 0; t < kDecMaxSteps; ++t) { yacc[t][0] = 0.f; yacc[t][1] = 0.f; yacc[t][2] = 0.f; yacc[t][3] = 0.f; }
      }
      // fp8 merged parts (two sub-blocks = 16 act columns in one part): ONE pass whose MMAs use all 16 k slots -- lane quarters 0 / 1
      // feed sub-block 0's columns 0-3 / 4-7, quarters 2 / 3 sub-block 1's
      const bool mg = F8 && g.merge != 0 && g.n_sb == 2;
      // bf16 units of two sub-blocks: their two down parts (consecutive in the ring) feed ONE pass whose MMAs use all 16 k slots
      // (k 0-7 = sub-block 0's act columns, k 8-15 = sub-block 1's) instead of two passes with half of K zero
      const bool pair = kMma && g.n_sb == 2;
      const int n_pass = (mg || pair) ? 1 : g.n_sb;
      for (int sb = 0; sb < n_pass; ++sb) {
      if (sb > 0) mbar_wait(ring.full0 + 8u * rp.s, rp.ph);
      const uint32_t pbase = ring.slot0 + (uint32_t)rp.s * ring.stride;
      const int sbx = mg ? (lane & 3) >> 1 : sb;                // sub-block this lane's operands come from
      const uint32_t dbase = pbase + (mg ? (uint32_t)sbx * (uint32_t)g.sub_bytes : 0u);
      store_part(DecPart{2, sb, s});
      const AT* act = reinterpret_cast<const AT*>(fs.act[par][sbx]);
      if constexpr (F8) {
        // a down core is 8 outputs x 8 act columns (64 bytes): lane quarters 0 / 1 hold columns 0-3 / 4-7 of outputs g and g + 8 and
        // feed the k slots {2q, 2q+1, 2q+8, 2q+9}; unmerged, quarters 2 / 3 contribute zeros (8 columns, 16 slots)
        const int tq = lane & 3;
        const bool on = mg || tq < 2;
        const uint2 bv = *reinterpret_cast<const uint2*>(reinterpret_cast<const __half*>(act) + col * 8 + (tq & 1) * 4);
        const uint32_t b0 = on ? bv.x : 0u, b1 = on ? bv.y : 0u;
        const uint32_t abase = dbase + (uint32_t)(warp * g.steps) * 128u + (uint32_t)(lane >> 2) * 8u + (uint32_t)(tq & 1) * 4u;
#pragma unroll
        for (int t0 = 0; t0 < kDecMaxSteps; t0 += 4) {
          if (t0 < g.steps) {
            uint32_t lo[4], hi[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
              lo[j] = lds_u32(abase + (uint32_t)(t0 + j) * 128u);
              hi[j] = lds_u32(abase + (uint32_t)(t0 + j) * 128u + 64u);
            }
#pragma unroll
            for (int j = 0; j < 4; ++j) {
              const uint32_t l = lo[j], h = hi[j];             // (quarters 2 / 3 re-read quarter 0 / 1's finite codes against B = 0)
              mma_f16_16816(yacc[t0 + j], cvt_e4m3x2_f16x2((uint16_t)l), cvt_e4m3x2_f16x2((uint16_t)h), cvt_e4m3x2_f16x2((uint16_t)(l >> 16)),
                            cvt_e4m3x2_f16x2((uint16_t)(h >> 16)), b0, b1);
            }
          }
        }
        float s2v[kDecMaxSteps / 8];                           // block scales of this warp's output blocks (read before the slot is released)
        if (sb == n_pass - 1) {
#pragma unroll
          for (int i = 0; i < kDecMaxSteps / 8; ++i)
            s2v[i] = i * 8 < g.steps ? lds_f32(pbase + (uint32_t)g.part_bytes + (uint32_t)(warp * (g.steps >> 3) + i) * 4u) : 0.f;
        }
        release();
        if (sb == n_pass - 1) {
          const int j0 = s * g.slab + warp * (g.slab >> 3) + col;
          float* p0 = a.partial + ((size_t)(pos0 + kq) * g.n_chunks + c) * g.d + j0;
          float* p1 = p0 + (size_t)g.n_chunks * g.d;
          if (kq < cnt) {                                      // (cnt is uniform over the warp: with one token only quarter 0 stores)
            const float as0 = fs.ascale[par][kq];
            const float sc[kDecMaxSteps / 8] = {s2v[0] * as0, s2v[1] * as0};
#pragma unroll
            for (int t = 0; t < kDecMaxSteps; ++t)
              if (t < g.steps) { p0[t * 16] = yacc[t][0] * sc[t >> 3]; p0[t * 16 + 8] = yacc[t][2] * sc[t >> 3]; }
          }
          if (cnt > 1 && kq + 1 < cnt) {
            const float as1 = fs.ascale[par][kq + 1];
            const float sc[kDecMaxSteps / 8] = {s2v[0] * as1, s2v[1] * as1};
#pragma unroll
            for (int t = 0; t < kDecMaxSteps; ++t)
              if (t < g.steps) { p1[t * 16] = yacc[t][1] * sc[t >> 3]; p1[t * 16 + 8] = yacc[t][3] * sc[t >> 3]; }
          }
        }
      } else if constexpr (kMma) {
        if (pair) {
          // A[j][i]: 16 outputs j x 16 act columns i (matrices 0, 1 from sub-block 0's part, 2, 3 from sub-block 1's); B[i][n] = a[n][i]
          DecRingPos rp1 = rp;
          ring_advance(ring, rp1);
          mbar_wait(ring.full0 + 8u * rp1.s, rp1.ph);
          const uint32_t d1base = ring.slot0 + (uint32_t)rp1.s * ring.stride;
          store_part(DecPart{2, 1, s}, rp1.s);
          const AT* act1 = reinterpret_cast<const AT*>(fs.act[par][1]);
          const uint32_t b0 = *reinterpret_cast<const uint32_t*>(act + col * 8 + kq), b1 = *reinterpret_cast<const uint32_t*>(act1 + col * 8 + kq);
          const uint32_t abase = ((lane >> 4) ? d1base : dbase) + (uint32_t)(lane & 7) * 16u + (uint32_t)((lane >> 3) & 1) * 128u +
                                 (uint32_t)(warp * g.steps) * 256u;
#pragma unroll
          for (int t0 = 0; t0 < kDecMaxSteps; t0 += 4) {      // four output tiles per batch: loads first, then the MMAs
            if (t0 < g.steps) {
              uint32_t af[4][4];
#pragma unroll
              for (int j = 0; j < 4; ++j)
                if (t0 + j < g.steps) ldmatrix_x4(af[j][0], af[j][1], af[j][2], af[j][3], abase + (uint32_t)(t0 + j) * 256u);
#pragma unroll
              for (int j = 0; j < 4; ++j)
                if (t0 + j < g.steps) mma_bf16_16816(yacc[t0 + j], af[j][0], af[j][1], af[j][2], af[j][3], b0, b1);
            }
          }
          release();                                           // sub-block 0's part
        } else {
        // A[j][i]: 16 outputs j x (8 act columns i, upper half of K zero); B[i][n] = a[n][i]
        const uint32_t b0 = *reinterpret_cast<const uint32_t*>(act + col * 8 + kq);
        const uint32_t abase = dbase + (uint32_t)(lane & 7) * 16u + (uint32_t)((lane >> 3) & 1) * 128u + (uint32_t)(warp * g.steps) * 256u;
#pragma unroll
        for (int t0 = 0; t0 < kDecMaxSteps; t0 += 4) {        // four output tiles per batch: loads first, then the MMAs
          if (t0 < g.steps) {
            uint32_t af[4][2];
#pragma unroll
            for (int j = 0; j < 4; ++j)
              if (t0 + j < g.steps) ldmatrix_x2(af[j][0], af[j][1], abase + (uint32_t)(t0 + j) * 256u);
#pragma unroll
            for (int j = 0; j < 4; ++j)
              if (t0 + j < g.steps) mma_bf16_16816(yacc[t0 + j], af[j][0], af[j][1], 0u, 0u, b0, 0u);
          }
        }
        }
        release();
        if (sb == n_pass - 1) {
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
      } else {
        // fp32: thread owns outputs j = tid, tid + 256, ... of the slab; fp32 models use one sub-block per unit, so the sum over
        // the 8 act columns is complete here: i ascending, fmaf from 0.f
        const uint32_t half = (uint32_t)g.part_bytes / 2;
        for (int jj = tid; jj < g.slab; jj += kDecConsumers) {
          float wv[8];
          const uint32_t addr = dbase + (uint32_t)(jj >> 3) * 128u + (uint32_t)(jj & 7) * 16u;
          asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(wv[0]), "=f"(wv[1]), "=f"(wv[2]), "=f"(wv[3]) : "r"(addr));
          asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(wv[4]), "=f"(wv[5]), "=f"(wv[6]), "=f"(wv[7]) : "r"(addr + half));
          for (int n = 0; n < cnt; ++n) {
            float acc = 0.f;
#pragma unroll
            for (int i = 0; i < 8; ++i) acc = fmaf(wv[i], to_f32<AT>(act[n * 8 + i]), acc);
            a.partial[((size_t)(pos0 + n) * g.n_chunks + c) * g.d + s * g.slab + jj] = acc;
          }
        }
        release();
      }
      }
      if (s == g.n_slab - 1) ++d_seq;
    }
  }
  if (a.master != nullptr && tid == 0) bulk_wait0();     // this CTA's slot fills are complete before the next grid-wide barrier
}

}  // namespace wisp
