// decode_kernels.cuh -- the decode hot path (a1-a5) of one token batch (n_tokens <= 8).
//
// Fused form (WISP_FETCH_FUSED, E <= 256): ONE persistent cooperative kernel per token batch, one CTA per SM, the whole
// stack of layers inside the launch.  The paper runs the paging decision in Python on the host between kernels and names
// that its overhead; here the whole chain stays on the chip with ONE grid-wide barrier per layer (C) and one
// data-carrying reduction (the logit accumulators count their own contributions, decode_combine.cuh):
//
//   route  every CTA: logits of this layer (bias + the int64 accumulator filled by the previous combine), top-k by warp
//          arg-max (router.cuh), Algorithm 1 -- the one-warp hit fast path, or plan_compute when the step
//          faults / overflows (residency.cuh) -- computed redundantly and deterministically per CTA; CTA 0 is the writer of
//          pi, pi^-1, tau, f, counters, trace
//   ffn    fused gate/up/SwiGLU/down per work unit (decode_ffn.cuh), units handed out by an atomic ticket, misses read
//          from the mapped pinned master and written into their victim slot on the way (Alg. 1 line 6)      -> barrier C
//   comb   16-column slices over the grid: ordered combine + residual -> x_{l+1}; partial router logits of layer l+1 into
//          the int64 accumulators (decode_combine.cuh); no barrier: the next route step polls the accumulator words until each
//          carries all its contributions, and one warp waits for the x-ready counter and reloads x_{l+1} (4 KiB per token)
// An overflowing step (|R| > C) adds one barrier per extra wave (the next wave's fills reuse slots).
//
// Split form (MEMCPY / ZEROCOPY contexts, E > 256, event timing of kernel classes): the same device functions as four
// launches per layer (logits, plan, ffn per wave, combine) with the demand fetch between plan and ffn, so every fetch path
// gives the same bits (parity (b)).
#pragma once
#include "common.cuh"
#include "decode_combine.cuh"
#include "decode_ffn.cuh"
#include "residency.cuh"
#include "router.cuh"

namespace wisp {

constexpr int kPersistMaxExperts = 256;     // plan capacity of the fused kernel (larger E -> split form)
constexpr int kDecPhases = 6;               // route, plan, prefetch of the next layer's state, ffn, ffn of layers with misses, combine
constexpr unsigned kGridBarrierSpinLimit = 1u << 24;
constexpr int kCombineBatch = 4;            // tokens whose slices of one column block a CTA combines in one pass

struct DecodeArgs {
  int L, E, k, d, dff, T, C, policy;
  int wave_order;               // wisp_wave_order (G25)
  int layer_lo, layer_hi;
  int residual;                 // 1: x_{l+1} = x_l + y_l chained, `out` = x_hi; 0: out = y (one layer)
  const char* pool;
  const char* const* masters;   // device array [L] of mapped pinned master pointers
  unsigned long long blob_bytes;
  const char* router_wt;        // [L][d][E] model dtype (transposed router weights)
  const float* router_bias;     // [L][E]
  int *pi, *pi_inv;
  u64 *tau, *freq, *scal, *last_pos, *hist;
  float* logits;                // [T][E] (test surface: wisp_last_logits)
  int* ids;                     // [L][max_tokens*k]
  float* topw;
  int max_tokens;
  float* partial;               // P [pair position][NC][d] fp32
  long long* zfix;              // [2][kZfixCopies][kDecodeMaxTokens][E] int64 logit accumulators, all zero between launches
  unsigned* sync;               // [0] grid barrier counter, [1..2] unit tickets, [3] x-ready counter (slices of x written so far); zero at launch
  const void* x_in;             // input of layer_lo, [T][d]
  void* xbuf[2];                // intermediate hidden states
  void* out;                    // [T][d]
  volatile int* err;            // mapped host flag: set to 1 if a grid barrier timed out
  wisp_trace_event* trace;
  u64* trace_ctr;
  u64 trace_cap;
  int trace_on, track;
  u64* phase_ns;                // nullable: [kDecPhases + 2] globaltimer ns summed by the last CTA, then counts of hit / miss layers
};

// The per-layer plan in shared memory (same fields as PlanPtrs).
struct DecPlan {
  int hdr[4];
  int entry_expert[kPersistMaxExperts], entry_slot[kPersistMaxExperts], entry_miss[kPersistMaxExperts];
  int exp_count[kPersistMaxExperts], exp_offset[kPersistMaxExperts + 1];
  int pair_list[kDecodeMaxTokens * kMaxTopK], pair_pos[kDecodeMaxTokens * kMaxTopK];
  int unit_entry[kPersistMaxExperts];
};
__device__ __forceinline__ PlanPtrs plan_ptrs_of(DecPlan& pl) {
  PlanPtrs pp;
  pp.hdr = pl.hdr; pp.entry_expert = pl.entry_expert; pp.entry_slot = pl.entry_slot; pp.entry_miss = pl.entry_miss;
  pp.exp_count = pl.exp_count; pp.exp_offset = pl.exp_offset; pp.pair_list = pl.pair_list;
  pp.unit_entry = pl.unit_entry; pp.pair_pos = pl.pair_pos;
  return pp;
}

__device__ __forceinline__ LayerState layer_state_of(const DecodeArgs& a, int l) {
  LayerState st;
  const size_t E = a.E;
  st.pi = a.pi + l * E; st.pi_inv = a.pi_inv + l * E; st.tau = a.tau + l * E; st.freq = a.freq + l * E;
  st.scal = a.scal + (size_t)l * 8; st.last_pos = a.last_pos + l * E; st.hist = a.hist + l * (E + 2);
  return st;
}

// Barrier over all CTAs, taken by the 256 consumer threads of each (named barrier 1).  `gen` counts the arrivals expected so
// far.  Returns false in every thread of the CTA if the barrier timed out (another CTA died): the caller leaves the kernel,
// and the host reports WISP_ECUDA from the flag.
__device__ __forceinline__ bool grid_barrier(unsigned* ctr, unsigned& gen, volatile int* err, int* s_abort) {
  gen += gridDim.x;
  asm volatile("bar.sync 1, 256;" ::: "memory");
  if (threadIdx.x == 0) {
    // release: the CTA's writes (ordered before this thread by the bar.sync above) become visible at gpu scope before the
    // arrival; acquire: each poll is LDG.STRONG.GPU + CCTL.IVALL, so this SM's L1 holds no stale line afterwards.
    red_release_add(ctr, 1u);
    unsigned spins = 0;
    while (ld_acquire(ctr) < gen) {
      // the flag lives in mapped host memory (a read crosses the host link): look at it only once in a while
      if (++spins > kGridBarrierSpinLimit || ((spins & 0xfffu) == 0u && *err)) { *err = 1; *s_abort = 1; break; }
    }
  }
  asm volatile("bar.sync 1, 256;" ::: "memory");
  return *reinterpret_cast<volatile int*>(s_abort) == 0;
}

// Shared state of one decode CTA besides the FFN dataflow (static shared memory of the fused kernel).
struct DecShared {
  unsigned long long go;                                  // the plan of the next wave exists: the producer may stream
  unsigned long long wpre;                                // the next layer's router-weight slice has landed in shared memory
  unsigned long long xbar;                                // x_l has landed in shared memory (bulk copies issued by warp 7)
  alignas(16) float y[kCombineBatch * kMaxTopK * kSliceCols];   // combine: per-rank sums of up to kCombineBatch slices
  float xn[kCombineBatch * kSliceCols];
  int zexp[kZfixCopies];                                  // partials a complete accumulator word of copy c carries (per token and layer)
  int ids[kDecodeMaxTokens * kMaxTopK];
  float w[kDecodeMaxTokens * kMaxTopK];
  DecPlan pl;
};

// MULTI: the launch has more than one token (adds the batched combine; the one-token instantiation keeps its registers).
template <typename T, bool F8, bool MULTI>
__global__ void __launch_bounds__(kDecThreads, 1) decode_fused_kernel(const DecodeArgs a, const DecodeGeom g, int n_slots, int xs_pitch,
                                                                      int pre_off, int ring_off) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  __shared__ __align__(16) DecShared ds;
  __shared__ __align__(16) DecFfnShared fs;
  __shared__ PlanShared<kPersistMaxExperts> sh;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  DecRing ring;
  ring.slot0 = smem_u32(smem_raw) + (uint32_t)ring_off; ring.full0 = smem_u32(fs.full); ring.empty0 = smem_u32(fs.empty);
  ring.n_slots = n_slots; ring.stride = g.slot_bytes;
  if (tid == 0) {
    mbar_init(smem_u32(&ds.go), 1);
    mbar_init(smem_u32(&ds.wpre), 1);
    mbar_init(smem_u32(&ds.xbar), 1);
    dec_ffn_shared_init(fs, ring);
  }
  __syncthreads();
  DecRingPos rp{0, 0u};
  const int E = a.E, k = a.k, d = a.d, T_ = a.T, C = a.C;
  const PlanPtrs pp = plan_ptrs_of(ds.pl);
  DecodeFfnArgs fa{};
  fa.slot_stride = (unsigned long long)a.L * a.blob_bytes; fa.blob_bytes = a.blob_bytes; fa.k = k; fa.inv_k = 1.0f / (float)k;
  fa.partial = a.partial;

  if (warp == kDecWarps + 1) {                           // ===================== reducer warp =====================
    decode_reduce<T, F8>(g, fs, lane);
    return;
  }
  if (warp == kDecWarps) {
    // ===================== producer warp (one lane): streams every wave's units as soon as its plan exists ==========
    if (lane != 0) return;
    const uint64_t pol = l2_evict_first_policy();
    unsigned qseq = 0;                                   // waves started so far (all layers)
    for (int l = a.layer_lo; l < a.layer_hi; ++l) {
      fa.layer_base = a.pool + (size_t)l * a.blob_bytes;
      fa.master = a.masters[l];
      int n_waves = 1;
      for (int w = 0; w < n_waves; ++w, ++qseq) {
        if (!mbar_wait_or_abort(smem_u32(&ds.go), qseq & 1u, &fs.abort)) return;
        n_waves = ds.pl.hdr[0];
        const int nR = ds.pl.hdr[1], lo = w * C, nw = min(nR, lo + C) - lo;
        fa.ticket = a.sync + 1 + (qseq & 1u);
        decode_produce<F8>(fa, g, pp, fs, ring, rp, lo, nw, pol);
        if (fs.abort) return;
      }
    }
    return;
  }

  // ===================== consumer warps =====================
  const bool writer = blockIdx.x == 0;
  // the timing CTA is not the writer and owns a combine slice (CTA 1); its route stamp includes the wait for the accumulators
  const bool timing = blockIdx.x == (gridDim.x > 1 ? 1u : 0u) && tid == 0 && a.phase_ns != nullptr;
  u64 t_prev = timing ? globaltimer_ns() : 0ull;
  auto stamp = [&](int phase) {
    if (timing) { const u64 t = globaltimer_ns(); atomicAdd(a.phase_ns + phase, t - t_prev); t_prev = t; }   // RED: no round trip
  };
  unsigned gen = 0, qseq = 0, gu_seq = 0, d_seq = 0;
  const uint32_t w_off = (uint32_t)((E * sizeof(float) + 127) & ~(size_t)127);   // staged region: [router bias of the next layer][weight slice]
  T* xs = reinterpret_cast<T*>(smem_raw);               // current hidden state, [T][xs_pitch], in EVERY CTA
  __half* xh = reinterpret_cast<__half*>(smem_raw + (((size_t)a.T * xs_pitch * sizeof(T) + 127) & ~(size_t)127));   // fp8 experts: f16 copy
  auto load_xs = [&](const void* src_) {
    const int vec_row = d * (int)sizeof(T) / 16;
    for (int i = tid; i < T_ * vec_row; i += kDecConsumers) {
      const int t = i / vec_row, c = i % vec_row;
      reinterpret_cast<uint4*>(xs + (size_t)t * xs_pitch)[c] = __ldcg(reinterpret_cast<const uint4*>(src_) + i);
    }
  };
  const int n_slices = T_ * (d / kSliceCols);
  const size_t zplane = zfix_plane(E);
  load_xs(a.x_in);
  if (tid < kZfixCopies) {
    int n = 0;
    for (int jb = 0; jb < d / kSliceCols; ++jb) n += ((jb % (int)gridDim.x) % kZfixCopies) == tid;
    ds.zexp[tid] = n;
  }
  plan_load<kPersistMaxExperts>(sh, layer_state_of(a, a.layer_lo), E, C);
  asm volatile("bar.sync 1, 256;" ::: "memory");
  // logits of the first layer: the same 16-column slices the combine uses for every later layer
  {
    const T* wrt = reinterpret_cast<const T*>(a.router_wt) + (size_t)a.layer_lo * d * E;
    // (the combine's mapping: CTA b owns the column blocks b, b + grid, ... of every token, so a copy receives ds.zexp[c] partials)
    for (int jb = blockIdx.x; jb < d / kSliceCols; jb += gridDim.x)
      for (int t = 0; t < T_; ++t) {
        const int j0 = jb * kSliceCols;
        if (tid < kSliceCols) ds.xn[tid] = to_f32<T>(xs[(size_t)t * xs_pitch + j0 + tid]);
        asm volatile("bar.sync 1, 256;" ::: "memory");
        slice_logits<T>(wrt + (size_t)j0 * E, ds.xn, E, a.zfix + ((size_t)(a.layer_lo & 1) * kZfixCopies + (blockIdx.x % kZfixCopies)) * zplane + (size_t)t * E, tid, kDecConsumers);
        asm volatile("bar.sync 1, 256;" ::: "memory");
      }
  }
  if (!grid_barrier(a.sync, gen, a.err, &fs.abort)) return;

  for (int l = a.layer_lo; l < a.layer_hi; ++l) {
    const LayerState st = layer_state_of(a, l);
    const bool last = l == a.layer_hi - 1;
    long long* zf_l = a.zfix + (size_t)(l & 1) * kZfixCopies * zplane;        // copy 0 of this layer's accumulators

    // ---- route: logits -> top-k (one warp per token); the other threads' loads of x_l (written by the previous layer's
    // combine) are in flight meanwhile ----
    const bool reload = l > a.layer_lo;
    const bool split = T_ * k <= kDecConsumers - 32;           // warp 7 loads x while warps 0-6 select (else: all select, then warp 7 loads)
    auto reload_x = [&]() {
      // ---- warp 7: x_l.  The previous combine's slices count themselves into the x-ready word after a gpu-scope fence ----
      if (reload) {
        if (lane == 0) {
          const unsigned want = (unsigned)(l - a.layer_lo) * (unsigned)n_slices;
          unsigned spins = 0;
          while (ld_acquire(a.sync + 3) < want)
            if (++spins > kGridBarrierSpinLimit || ((spins & 0xfffu) == 0u && *a.err)) { *a.err = 1; fs.abort = 1; break; }
        }
        if constexpr (MULTI && !F8) {
          // bf16 batches: one bulk copy per token row (rows are padded in shared memory): all in flight together, one L2 round trip
          // whatever T is.  (One token, and fp8 experts -- whose f16 staging pass follows -- measured faster with the loads below.)
          if (lane == 0 && !fs.abort) {
            asm volatile("fence.proxy.async;" ::: "memory");    // the acquire above orders the rows' generic-proxy writes before these reads
            const uint32_t row_bytes = (uint32_t)(d * sizeof(T));
            const char* x_src = reinterpret_cast<const char*>(a.xbuf[(l - 1 - a.layer_lo) & 1]);
            mbar_expect_tx(smem_u32(&ds.xbar), (uint32_t)T_ * row_bytes);
            for (int t = 0; t < T_; ++t)
              bulk_g2s_nohint(smem_u32(xs) + (uint32_t)t * (uint32_t)(xs_pitch * sizeof(T)), x_src + (size_t)t * row_bytes, row_bytes, smem_u32(&ds.xbar));
          }
          __syncwarp();
          mbar_wait_or_abort(smem_u32(&ds.xbar), (unsigned)(l - 1 - a.layer_lo) & 1u, &fs.abort);
        } else {
          __syncwarp();
          const uint4* x_src = reinterpret_cast<const uint4*>(a.xbuf[(l - 1 - a.layer_lo) & 1]);
          const int vec_row = d * (int)sizeof(T) / 16, xs_vec = T_ * vec_row;
          for (int v0 = lane; v0 < xs_vec; v0 += 32 * 8) {
            uint4 xr[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) xr[i] = __ldcg(x_src + min(v0 + 32 * i, xs_vec - 1));
#pragma unroll
            for (int i = 0; i < 8; ++i) {
              const int v = v0 + 32 * i;
              if (v < xs_vec) reinterpret_cast<uint4*>(xs + (size_t)(v / vec_row) * xs_pitch)[v % vec_row] = xr[i];
            }
          }
        }
      }
    };
    if (split && warp == kDecWarps - 1) {
      reload_x();
    } else {
      // ---- warps 0-6: logits -> top-k.  Every accumulator word is polled until it carries all its partials ----
      const float* bias = a.router_bias + (size_t)l * E;
      if (reload) {                                            // staged in shared memory during the previous layer's FFN
        mbar_wait(smem_u32(&ds.wpre), (unsigned)(l - 1 - a.layer_lo) & 1u);
        bias = reinterpret_cast<const float*>(smem_raw + pre_off);
      }
      float* zout = writer ? a.logits : nullptr;               // test surface: wisp_last_logits
      auto zf = [&](int t, int e) {
        const long long* w0 = zf_l + (size_t)t * E + e;
        long long v[kZfixCopies];
        unsigned spins = 0;
        while (true) {
          bool done = true;
#pragma unroll
          for (int c = 0; c < kZfixCopies; ++c) v[c] = ld_relaxed_s64(w0 + c * zplane);
#pragma unroll
          for (int c = 0; c < kZfixCopies; ++c) done = done && zfix_count(v[c]) == ds.zexp[c];
          if (done) break;
          if (++spins > kGridBarrierSpinLimit || ((spins & 0xfffu) == 0u && (*a.err || fs.abort))) { *a.err = 1; fs.abort = 1; break; }
        }
        long long sum = 0;
#pragma unroll
        for (int c = 0; c < kZfixCopies; ++c) sum += zfix_value(v[c]);
        const float z = logit_from_fix(sum, bias[e]);
        if (zout) zout[(size_t)t * E + e] = z;
        return z;
      };
      // (T * k <= 256 pairs: kDecodeMaxTokens * kMaxTopK; the FFN dataflow's scratch is idle between waves)
      if (split) topk_softmax_block(zf, T_, E, k, ds.ids, ds.w, reinterpret_cast<unsigned*>(&fs.red[0][0][0]), tid, kDecConsumers - 32, 2);
      else topk_softmax_block(zf, T_, E, k, ds.ids, ds.w, reinterpret_cast<unsigned*>(&fs.red[0][0][0]), tid, kDecConsumers, 1);
    }
    if (!split && warp == kDecWarps - 1) reload_x();
    asm volatile("bar.sync 1, 256;" ::: "memory");
    if (fs.abort) return;                                      // a poll timed out: the host reports WISP_ECUDA
    if constexpr (F8)                                          // (the plan step's barriers order it before the consumers' reads)
      stage_xh(reinterpret_cast<const __nv_bfloat16*>(xs), xh, fs, T_, d, xs_pitch, tid, kDecConsumers,
               [] { asm volatile("bar.sync 1, 256;" ::: "memory"); });
    stamp(0);
    if (writer && tid < T_ * k) {
      const size_t off = (size_t)l * a.max_tokens * k;
      a.ids[off + tid] = ds.ids[tid];
      a.topw[off + tid] = ds.w[tid];
    }
    // ---- plan: Algorithm 1, redundantly in every CTA ----
    {
      PlanArgs pa;
      pa.ids = ds.ids; pa.n_pairs = T_ * k; pa.E = E; pa.C = C; pa.policy = a.policy; pa.layer = l;
      pa.st = st; pa.plan = pp; pa.host_plan = nullptr;
      pa.trace = a.trace; pa.trace_ctr = a.trace_ctr; pa.trace_cap = a.trace_cap; pa.trace_on = a.trace_on;
      pa.track = a.track; pa.build_pairs = 1; pa.wave_order = a.wave_order;
      if (warp == 0) {
        const bool fast = plan_fast_warp<kPersistMaxExperts>(pa, sh, writer, lane);
        if (lane == 0) ds.pl.hdr[0] = fast ? ds.pl.hdr[0] : -1;
      }
      asm volatile("bar.sync 1, 256;" ::: "memory");
      if (ds.pl.hdr[0] < 0) {
        asm volatile("bar.sync 1, 256;" ::: "memory");         // every thread has seen the flag before plan_compute rewrites hdr
        plan_compute<kPersistMaxExperts>(pa, sh, writer, 1);
      }
    }
    const int n_waves = ds.pl.hdr[0];
    const int miss_cls = ds.pl.hdr[2] > 0 ? 1 : 0;             // layers with misses are timed apart
    // this CTA's first combine slice is known now: its 16 rows of the NEXT layer's router weights (one contiguous block of
    // [d][E]) are staged in shared memory by a bulk copy while the FFN streams
    const bool pre = !last && (int)blockIdx.x < d / kSliceCols;
    if (tid == 0) {
      if (writer) a.sync[1 + ((qseq + 1) & 1u)] = 0u;          // ticket counter of the NEXT wave (idle since the wave before this one)
      mbar_arrive(smem_u32(&ds.go));                           // the producer may start streaming
      if (!last) {                                             // + the next layer's router bias (every CTA routes)
        const uint32_t wbytes = pre ? (uint32_t)(kSliceCols * E * sizeof(T)) : 0u, bbytes = (uint32_t)(E * sizeof(float));
        mbar_expect_tx(smem_u32(&ds.wpre), wbytes + bbytes);
        bulk_g2s_nohint(smem_u32(smem_raw) + (uint32_t)pre_off, a.router_bias + (size_t)(l + 1) * E, bbytes, smem_u32(&ds.wpre));
        if (pre) {
          const T* src = reinterpret_cast<const T*>(a.router_wt) + ((size_t)(l + 1) * d + (size_t)((int)blockIdx.x % (d / kSliceCols)) * kSliceCols) * E;
          bulk_g2s_nohint(smem_u32(smem_raw) + (uint32_t)pre_off + w_off, src, wbytes, smem_u32(&ds.wpre));
        }
      }
    }
    stamp(1);
    if (!last) plan_load<kPersistMaxExperts>(sh, layer_state_of(a, l + 1), E, C);   // stable until that layer's own plan
    stamp(2);
    if (timing) atomicAdd(a.phase_ns + kDecPhases + miss_cls, 1ull);

    // ---- ffn, wave by wave ----
    fa.layer_base = a.pool + (size_t)l * a.blob_bytes;
    fa.master = a.masters[l];
    for (int w = 0; w < n_waves; ++w, ++qseq) {
      if (w > 0) {
        if (!grid_barrier(a.sync, gen, a.err, &fs.abort)) return;   // the previous wave's slots may now be refilled
        if (tid == 0) {
          if (writer) a.sync[1 + ((qseq + 1) & 1u)] = 0u;
          mbar_arrive(smem_u32(&ds.go));
        }
      }
      fa.ticket = a.sync + 1 + (qseq & 1u);
      decode_consume<T, F8>(fa, g, pp, fs, ring, rp, gu_seq, d_seq, xs, xh, xs_pitch);
    }
    if (n_waves == 0) ++qseq;                                  // (cannot happen: n_tokens >= 1) keeps the producer in step
    if (!grid_barrier(a.sync, gen, a.err, &fs.abort)) return;  // C: every chunk partial of this layer is in place
    stamp(3 + miss_cls);

    // ---- combine (+ residual) and the next layer's logits, 16-column slices over the grid ----
    {
      if (writer)                                                // consumed above by every CTA
        for (int c = 0; c < kZfixCopies; ++c)
          for (int i = tid; i < T_ * E; i += kDecConsumers) zf_l[c * zplane + i] = 0ll;
      CombineArgs ca;
      ca.partial = a.partial; ca.n_chunks = g.n_chunks; ca.d = d; ca.k = k; ca.topw = ds.w; ca.pair_pos = ds.pl.pair_pos;
      T* xg = reinterpret_cast<T*>(last ? a.out : a.xbuf[(l - a.layer_lo) & 1]);
      const T* wrt = reinterpret_cast<const T*>(a.router_wt) + (size_t)(l + 1) * d * E;
      long long* zf_n = a.zfix + ((size_t)((l + 1) & 1) * kZfixCopies + (blockIdx.x % kZfixCopies)) * zplane;
      // CTA b owns the column blocks b, b + grid, ... of EVERY token: the tokens of a block are combined kCombineBatch at a time (their
      // partial loads in flight together) and share the block's 16 rows of router weights (staged for the CTA's first block)
      const int n_jb = d / kSliceCols;
      for (int jb = blockIdx.x; jb < n_jb; jb += gridDim.x) {
        const int j0 = jb * kSliceCols;
        const T* w16 = wrt + (size_t)j0 * E;
        if (!last && jb == (int)blockIdx.x) {
          mbar_wait(smem_u32(&ds.wpre), (unsigned)(l - a.layer_lo) & 1u);
          w16 = reinterpret_cast<const T*>(smem_raw + pre_off + w_off);
        }
        for (int t0 = 0; t0 < T_; t0 += MULTI ? kCombineBatch : 1) {
          const int ns = MULTI ? min(kCombineBatch, T_ - t0) : 1;
          const T* xres = a.residual ? xs : nullptr;
          if (!MULTI || ns == 1) {
            if (g.n_chunks <= 64) combine_slice<T, 8>(ca, t0, j0, xres ? xres + (size_t)t0 * xs_pitch : nullptr, xg + (size_t)t0 * d, fs.red[0][0], ds.y, ds.xn, 1);
            else combine_slice<T, 16>(ca, t0, j0, xres ? xres + (size_t)t0 * xs_pitch : nullptr, xg + (size_t)t0 * d, fs.red[0][0], ds.y, ds.xn, 1);
            if (!last && tid == 255) { __threadfence(); atomicAdd(a.sync + 3, 1u); }    // x slice visible at gpu scope, then counted (a thread with no logit adds at E <= 255)
            if (!last) slice_logits<T>(w16, ds.xn, E, zf_n + (size_t)t0 * E, tid, kDecConsumers);
          } else if constexpr (!MULTI) {
          } else if (ns == 2) {
            combine_tokens<T, 2, 6>(ca, t0, ns, j0, xres, xs_pitch, xg, fs.red[0][0], ds.y, ds.xn, 1);
            if (!last && tid == 255) { __threadfence(); atomicAdd(a.sync + 3, (unsigned)ns); }
            if (!last) slice_logits_multi<T, 2>(w16, ds.xn, ns, E, zf_n + (size_t)t0 * E, tid, kDecConsumers);
          } else {
            combine_tokens<T, kCombineBatch, 3>(ca, t0, ns, j0, xres, xs_pitch, xg, fs.red[0][0], ds.y, ds.xn, 1);
            if (!last && tid == 255) { __threadfence(); atomicAdd(a.sync + 3, (unsigned)ns); }
            if (!last) slice_logits_multi<T, kCombineBatch>(w16, ds.xn, ns, E, zf_n + (size_t)t0 * E, tid, kDecConsumers);
          }
        }
      }
    }
    stamp(5);
  }
  if (tid == 0) fs.final = 1;                                   // lets the reducer warp leave
}

// ===================== split form: the same steps as separate launches =====================

// logits: grid = any; adds the 16-column partial logits of x [T][d] into zfix[t][e].
template <typename T>
__global__ void __launch_bounds__(256) decode_logits_kernel(const T* __restrict__ x, const T* __restrict__ wrt, long long* zfix, int n_tokens,
                                                            int E, int d) {
  __shared__ float s_xn[kSliceCols];
  const int n_slices = n_tokens * (d / kSliceCols);
  for (int sl = blockIdx.x; sl < n_slices; sl += gridDim.x) {
    const int t = sl / (d / kSliceCols), j0 = (sl % (d / kSliceCols)) * kSliceCols;
    if (threadIdx.x < kSliceCols) s_xn[threadIdx.x] = to_f32<T>(x[(size_t)t * d + j0 + threadIdx.x]);
    __syncthreads();
    slice_logits<T>(wrt + (size_t)j0 * E, s_xn, E, zfix + (blockIdx.x % kZfixCopies) * zfix_plane(E) + (size_t)t * E, threadIdx.x, 256);
    __syncthreads();
  }
}

// plan: one CTA of NT threads (NT >= E): logits -> top-k -> Algorithm 1 -> plan in global memory; clears the accumulator.
template <int NT>
__global__ void __launch_bounds__(NT) decode_plan_kernel(PlanArgs a, long long* zfix, const float* __restrict__ bias, float* __restrict__ logits,
                                                         int* __restrict__ ids, float* __restrict__ topw, int n_tokens, int k) {
  __shared__ PlanShared<NT> sh;
  __shared__ int s_fast;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  plan_load<NT>(sh, a.st, a.E, a.C);
  if (warp < n_tokens) {
    const long long* zt = zfix + (size_t)warp * a.E;
    auto zf = [&](int e) { return logit_from_fix(zfix_sum(zt + e, zfix_plane(a.E)), bias[e]); };
    topk_softmax_warp<NT / 32>(zf, a.E, k, ids + warp * k, topw + warp * k, lane);
    for (int e = lane; e < a.E; e += 32) logits[(size_t)warp * a.E + e] = zf(e);
  }
  __syncthreads();
  for (int c = 0; c < kZfixCopies; ++c)
    for (int i = tid; i < n_tokens * a.E; i += NT) zfix[c * zfix_plane(a.E) + i] = 0ll;
  a.ids = ids;
  if (warp == 0) {
    const bool fast = plan_fast_warp<NT>(a, sh, true, lane);
    if (lane == 0) s_fast = fast;
  }
  __syncthreads();
  if (!s_fast) plan_compute<NT>(a, sh, /*writer=*/true, /*bar=*/0);
  else if (a.host_plan && tid == 0) {
    // the MEMCPY path reads the plan on the host: a hit-only step has nothing to fetch
    a.host_plan->n_ref = a.plan.hdr[1]; a.host_plan->n_miss = 0; a.host_plan->n_pairs = a.n_pairs;
    for (int i = 0; i < a.plan.hdr[1]; ++i) {
      a.host_plan->entry_expert[i] = a.plan.entry_expert[i]; a.host_plan->entry_slot[i] = a.plan.entry_slot[i]; a.host_plan->entry_miss[i] = 0;
    }
    __threadfence_system();
    a.host_plan->n_waves = a.plan.hdr[0];
  }
}

// ffn: one wave of the plan in global memory; grid = SM count; `ticket` is zero at launch.
template <typename T, bool F8>
__global__ void __launch_bounds__(kDecThreads, 1) decode_ffn_kernel(DecodeFfnArgs fa, const DecodeGeom g, PlanPtrs gp, int wave, int C, int E,
                                                                    int n_tokens, const T* __restrict__ x, int n_slots, int xs_pitch,
                                                                    int ring_off) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  __shared__ __align__(16) DecFfnShared fs;
  __shared__ DecPlan spl;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (wave >= gp.hdr[0]) return;
  DecRing ring;
  ring.slot0 = smem_u32(smem_raw) + (uint32_t)ring_off; ring.full0 = smem_u32(fs.full); ring.empty0 = smem_u32(fs.empty);
  ring.n_slots = n_slots; ring.stride = g.slot_bytes;
  if (tid == 0) dec_ffn_shared_init(fs, ring);
  // the plan -> shared memory (the consumers index it per part)
  const int nR = gp.hdr[1], n_pairs = gp.hdr[3];
  for (int i = tid; i < nR; i += kDecThreads) {
    spl.entry_expert[i] = gp.entry_expert[i]; spl.entry_slot[i] = gp.entry_slot[i]; spl.entry_miss[i] = gp.entry_miss[i];
    spl.unit_entry[i] = gp.unit_entry[i];
  }
  for (int i = tid; i < n_pairs; i += kDecThreads) spl.pair_list[i] = gp.pair_list[i];
  PlanPtrs pp = plan_ptrs_of(spl);
  pp.exp_count = gp.exp_count; pp.exp_offset = gp.exp_offset;     // indexed by expert id (E may exceed the shared capacity)
  T* xs = reinterpret_cast<T*>(smem_raw);
  {
    const int vec_row = g.d * (int)sizeof(T) / 16;
    for (int i = tid; i < n_tokens * vec_row; i += kDecThreads)
      reinterpret_cast<uint4*>(xs + (size_t)(i / vec_row) * xs_pitch)[i % vec_row] = reinterpret_cast<const uint4*>(x)[i];
  }
  __syncthreads();
  __half* xh = reinterpret_cast<__half*>(smem_raw + (((size_t)n_tokens * xs_pitch * sizeof(T) + 127) & ~(size_t)127));
  if constexpr (F8) {
    stage_xh(reinterpret_cast<const __nv_bfloat16*>(xs), xh, fs, n_tokens, g.d, xs_pitch, tid, kDecThreads, [] { __syncthreads(); });
    __syncthreads();
  }
  DecRingPos rp{0, 0u};
  fa.inv_k = 1.0f / (float)fa.k;
  const int lo = wave * C, nw = min(nR, lo + C) - lo;
  if (warp == kDecWarps + 1) {
    decode_reduce<T, F8>(g, fs, lane);
  } else if (warp == kDecWarps) {
    if (lane == 0) decode_produce<F8>(fa, g, pp, fs, ring, rp, lo, nw, l2_evict_first_policy());
  } else {
    unsigned gu_seq = 0, d_seq = 0;
    decode_consume<T, F8>(fa, g, pp, fs, ring, rp, gu_seq, d_seq, xs, xh, xs_pitch);
    asm volatile("bar.sync 1, 256;" ::: "memory");
    if (tid == 0) fs.final = 1;
  }
}

// combine: grid = any; out (and, with x_res, the residual successor) from the chunk partials of all waves.
template <typename T>
__global__ void __launch_bounds__(256) decode_combine_kernel(CombineArgs ca, const T* __restrict__ x_res, T* __restrict__ dst, int n_tokens) {
  __shared__ __align__(16) float s_yg[8 * 8 * kSliceCols];
  __shared__ __align__(16) float s_y[kMaxTopK * kSliceCols];
  __shared__ float s_xn[kSliceCols];
  const int n_slices = n_tokens * (ca.d / kSliceCols);
  for (int sl = blockIdx.x; sl < n_slices; sl += gridDim.x) {
    const int t = sl / (ca.d / kSliceCols), j0 = (sl % (ca.d / kSliceCols)) * kSliceCols;
    combine_slice<T>(ca, t, j0, x_res ? x_res + (size_t)t * ca.d : nullptr, dst + (size_t)t * ca.d, s_yg, s_y, s_xn, 0);
  }
}

template <typename T>
__global__ void __launch_bounds__(256) residual_add_kernel(const T* __restrict__ x, const T* __restrict__ y,
                                                           T* __restrict__ out, size_t n) {
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx < n) out[idx] = from_f32<T>(to_f32<T>(x[idx]) + to_f32<T>(y[idx]));
}

}  // namespace wisp
