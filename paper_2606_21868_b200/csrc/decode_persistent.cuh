// decode_persistent.cuh -- the whole decode hot path (a1-a5) of one token batch (n_tokens <= 8) as ONE persistent
// cooperative kernel: one CTA per SM, layers lo..hi-1 back to back, grid-wide barriers between dependent phases.
//
// Why: at the Qwen3-30B-A3B shape one layer streams only 72 MiB (11.5 us at the measured 6.5 TB/s), so kernel
// boundaries, launch ramps and the router -> top-k -> Algorithm 1 dependency chain cost more than the FFN itself
// (profiles/r01_v1: 7 launches and 58 us per layer).  The paper names exactly this overhead (policy in Python on
// the hot path, no CUDA graphs).  Here the chain stays on chip:
//
//   phase R  router logits            warps of all CTAs take expert rows (router_row_warp)        -> barrier B
//   phase P  top-k + Algorithm 1      EVERY CTA computes the same plan redundantly in shared memory (integer work,
//                   deterministic); CTA 0 is the writer of pi, pi^-1, tau, f, counters and trace
//   phase G  gate/up + SwiGLU         TMA ring (ffn_stream.cuh); a miss is read from the mapped pinned master and
//   phase D  down                     written into its victim slot on the way (Alg. 1 line 6).  The
//                                     producer warp runs ahead: down tiles land in the ring while the CTA waits at
//                                     barrier C for the other CTAs' act rows                      -> barriers C, D
//   phase X  combine (+ residual)     split over the grid (combine_elem's sum), x_{l+1} via global memory -> barrier E,
//                                     then every CTA reloads x_{l+1} into its shared memory
//
// Every arithmetic step calls the same device function as the multi-kernel path (router_row_warp,
// topk_softmax_block, plan_compute, stream_consume, combine_elem), so both paths give the same bits (parity (b)).
#pragma once
#include "common.cuh"
#include "ffn_stream.cuh"
#include "residency.cuh"
#include "router.cuh"

namespace wisp {

constexpr int kPersistMaxExperts = 256;     // plan capacity of the persistent kernel (larger E -> multi-kernel path)
constexpr int kPersistPhases = 9;           // router, top-k, plan, next-layer prefetch, gate_up, down, combine, gate_up / down of layers with misses
constexpr unsigned kGridBarrierSpinLimit = 1u << 26;

struct PersistArgs {
  int L, E, k, d, dff, T, C, policy;
  int wave_order;               // wisp_wave_order (G25)
  int layer_lo, layer_hi;
  int residual;                 // 1: x_{l+1} = x_l + y_l chained through xbuf, `out` = x_hi; 0: out = y (one layer)
  int fused;                    // misses are read from the mapped master by the FFN producer
  const char* pool;
  const char* const* masters;   // device array [L] of mapped pinned master pointers
  unsigned long long blob_bytes;
  const char* router_w;         // [L][E][d] model dtype
  const float* router_bias;     // [L][E]
  int *pi, *pi_inv;
  u64 *tau, *freq, *scal, *last_pos, *hist;
  float* logits;                // [T][E]
  int* ids;                     // [L][max_tokens*k]
  float* topw;
  int max_tokens;
  float* act;                   // [T*k][dff] fp32
  float* ystage;                // [T*k][d] fp32
  const void* x_in;             // input of layer_lo, [T][d]
  void* xbuf[2];                // intermediate hidden states (stack mode)
  void* out;                    // [T][d]
  unsigned* gbar;               // grid barrier counter, zero at launch
  int* err;                     // set to 1 if a grid barrier timed out
  wisp_trace_event* trace;
  u64* trace_ctr;
  u64 trace_cap;
  int trace_on, track;
  u64* phase_ns;                // nullable: [kPersistPhases] globaltimer ns summed by CTA 0
};

struct PersistPlan {            // the per-layer plan in shared memory (same fields as PlanPtrs)
  int hdr[4];
  int entry_expert[kPersistMaxExperts], entry_slot[kPersistMaxExperts], entry_miss[kPersistMaxExperts];
  int exp_count[kPersistMaxExperts], exp_offset[kPersistMaxExperts + 1];
  int pair_list[kDecodeMaxTokens * kMaxTopK];
};

__device__ __forceinline__ LayerState layer_state_of(const PersistArgs& a, int l) {
  LayerState st;
  const size_t E = a.E;
  st.pi = a.pi + l * E; st.pi_inv = a.pi_inv + l * E; st.tau = a.tau + l * E; st.freq = a.freq + l * E;
  st.scal = a.scal + (size_t)l * 8; st.last_pos = a.last_pos + l * E; st.hist = a.hist + l * (E + 2);
  return st;
}

__device__ __forceinline__ void l2_prefetch(const void* p, uint32_t bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}

__device__ __forceinline__ u64 globaltimer_ns() {
  u64 t;
  asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
  return t;
}

// Barrier over all CTAs, taken by the 256 consumer threads of each (named barrier 1).  `gen` counts arrivals expected.
__device__ __forceinline__ void grid_barrier(unsigned* ctr, unsigned& gen, int* err) {
  gen += gridDim.x;
  asm volatile("bar.sync 1, 256;" ::: "memory");
  if (threadIdx.x == 0) {
    // release: the CTA's writes (ordered before this thread by the bar.sync above) become visible at gpu scope before the
    // arrival (SASS: MEMBAR.ALL.GPU + REDG.STRONG.GPU); acquire: each poll is LDG.STRONG.GPU + CCTL.IVALL, so this SM's L1
    // holds no stale line when the other threads pass the bar.sync below.  No return value, no trailing fence: 3.5 % faster
    // per token than __threadfence + atomicAdd + __threadfence.
    asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(ctr) : "memory");
    unsigned seen, spins = 0;
    do {
      asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(ctr) : "memory");
      if (++spins > kGridBarrierSpinLimit) { *err = 1; break; }
    } while (seen < gen);
  }
  asm volatile("bar.sync 1, 256;" ::: "memory");
}

template <typename T, int NP>
__global__ void __launch_bounds__(kStreamThreads, 1) decode_persistent_kernel(const PersistArgs a, const StreamGeom ggu,
                                                                              const StreamGeom gdn, int n_stages, int stage_stride,
                                                                              int xs_bytes, int rw_bytes) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  __shared__ __align__(8) unsigned long long s_full[kStreamMaxStages], s_empty[kStreamMaxStages], s_plan_ready, s_rw_bar;
  __shared__ float s_red[StreamRed<NP>::kFloats];
  __shared__ PlanShared<kPersistMaxExperts> sh;
  __shared__ PersistPlan pl;
  __shared__ float s_z[NP * kPersistMaxExperts];   // logits, rows packed E apart
  __shared__ float s_selz[NP * kMaxTopK];
  __shared__ int s_ids[NP * kMaxTopK];
  __shared__ float s_w[NP * kMaxTopK];

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  Ring ring;
  ring.stage0 = smem_u32(smem_raw) + (uint32_t)(xs_bytes + rw_bytes); ring.full0 = smem_u32(s_full); ring.empty0 = smem_u32(s_empty);
  ring.NS = n_stages; ring.stride = stage_stride;
  if (tid == 0) {
    mbar_init(smem_u32(&s_plan_ready), 1);
    mbar_init(smem_u32(&s_rw_bar), 1);
    ring_init(ring);
  }
  __syncthreads();
  RingPos rp{0, 0u};
  const int E = a.E, k = a.k, d = a.d, dff = a.dff, T_ = a.T, C = a.C;
  PlanPtrs pp;
  pp.hdr = pl.hdr; pp.entry_expert = pl.entry_expert; pp.entry_slot = pl.entry_slot; pp.entry_miss = pl.entry_miss;
  pp.exp_count = pl.exp_count; pp.exp_offset = pl.exp_offset; pp.pair_list = pl.pair_list;
  StreamArgs sa{};
  sa.plan = pp; sa.C = C; sa.pool = a.pool; sa.blob_bytes = a.blob_bytes; sa.L = a.L; sa.k = k; sa.pdl = 0;

  if (warp == kStreamConsumers / 32) {
    // ===================== producer warp: streams every layer's weight tiles as soon as its plan exists ==========
    const uint64_t pol = l2_evict_first_policy();
    for (int l = a.layer_lo; l < a.layer_hi; ++l) {
      mbar_wait(smem_u32(&s_plan_ready), (uint32_t)((l - a.layer_lo) & 1));
      sa.layer = l;
      sa.master = a.fused ? a.masters[l] : nullptr;
      const int n_waves = pl.hdr[0], nR = pl.hdr[1];
      for (int w = 0; w < n_waves; ++w) {
        const int lo = w * C, nw = min(nR, lo + C) - lo;
        {
          const long long U = (long long)nw * ggu.upe;
          stream_produce(sa, ggu, ring, rp, lo, (int)(U * blockIdx.x / gridDim.x), (int)(U * (blockIdx.x + 1) / gridDim.x), lane, pol);
        }
        {
          const long long U = (long long)nw * gdn.upe;
          stream_produce(sa, gdn, ring, rp, lo, (int)(U * blockIdx.x / gridDim.x), (int)(U * (blockIdx.x + 1) / gridDim.x), lane, pol);
        }
      }
    }
    return;
  }

  // ===================== consumer warps =====================
  const bool writer = blockIdx.x == 0;
  const bool timing = writer && tid == 0 && a.phase_ns != nullptr;
  u64 t_prev = timing ? globaltimer_ns() : 0ull;
  bool mute = false;    // probe builds: layers with misses are left out of the timeline
  auto stamp = [&](int phase) {
    if (timing) { const u64 t = globaltimer_ns(); if (!mute) a.phase_ns[phase] += t - t_prev; t_prev = t; }
  };
  unsigned gen = 0;
  int par = 0;
  plan_load<kPersistMaxExperts>(sh, layer_state_of(a, a.layer_lo), E, C);
  // The hidden state of the current layer lives in shared memory in EVERY CTA (xs, model dtype, [T][d]): the router
  // rows and the gate/up operand slices read it from there, and phase X recomputes x_{l+1} redundantly per CTA, so
  // no grid barrier and no global round trip separates a layer's combine from the next layer's router.
  T* xs = reinterpret_cast<T*>(smem_raw);
  {
    const uint4* src = reinterpret_cast<const uint4*>(a.x_in);
    uint4* dst = reinterpret_cast<uint4*>(xs);
    const int nvec = T_ * d * (int)sizeof(T) / 16;
    for (int i = tid; i < nvec; i += kStreamConsumers) dst[i] = src[i];
  }
  asm volatile("bar.sync 1, 256;" ::: "memory");
  // Router rows of this CTA (expert e = r * gridDim.x + blockIdx.x for warp r) are staged in shared memory by a TMA
  // bulk copy issued one layer ahead, so phase R starts from on-chip data; the bias rides along in a register.
  const int row_bytes = d * (int)sizeof(T);
  T* rw = reinterpret_cast<T*>(smem_raw + xs_bytes);
  const int my_e = warp * (int)gridDim.x + (int)blockIdx.x;               // this warp's expert row (if < E)
  int n_my_rows = 0;
  for (int r = 0; r < kStreamConsumers / 32; ++r) n_my_rows += (r * (int)gridDim.x + (int)blockIdx.x) < E && (r + 1) * row_bytes <= rw_bytes;
  const bool row_staged = my_e < E && (warp + 1) * row_bytes <= rw_bytes;
  float bias_next = 0.f;
  auto stage_router_rows = [&](int layer) {
    if (row_staged) bias_next = a.router_bias[(size_t)layer * E + my_e];
    if (tid == 0 && n_my_rows > 0) {
      mbar_expect_tx(smem_u32(&s_rw_bar), (uint32_t)(n_my_rows * row_bytes));
      for (int r = 0; r < n_my_rows; ++r)
        bulk_g2s_nohint(smem_u32(rw) + r * row_bytes, a.router_w + ((size_t)layer * E + r * gridDim.x + blockIdx.x) * row_bytes,
                        (uint32_t)row_bytes, smem_u32(&s_rw_bar));
    }
  };
  stage_router_rows(a.layer_lo);
  for (int l = a.layer_lo; l < a.layer_hi; ++l) {
    const T* x_l = xs;
    const LayerState st = layer_state_of(a, l);

    // ---- phase R: router logits (this layer's residency state is already in `sh`, its router rows in smem) ----
    {
      const float bias_cur = bias_next;
      if (row_staged) {
        mbar_wait(smem_u32(&s_rw_bar), (uint32_t)((l - a.layer_lo) & 1));
        for (int t0 = 0; t0 < T_; t0 += kRouterTokTile)
          router_row_warp<T>(x_l, rw + (size_t)warp * d, bias_cur, a.logits, my_e, t0, min(kRouterTokTile, T_ - t0), E, d, lane);
      }
      const T* wr = reinterpret_cast<const T*>(a.router_w) + (size_t)l * E * d;   // rows beyond the staging buffer: from global
      const float* bias = a.router_bias + (size_t)l * E;
      for (int e = my_e; e < E; e += (kStreamConsumers / 32) * gridDim.x)
        if (!(e == my_e && row_staged))
          for (int t0 = 0; t0 < T_; t0 += kRouterTokTile)
            router_row_warp<T>(x_l, wr + (size_t)e * d, bias[e], a.logits, e, t0, min(kRouterTokTile, T_ - t0), E, d, lane);
    }
    grid_barrier(a.gbar, gen, a.err);                                        // B: logits complete
    stamp(0);

    // ---- phase P: top-k + softmax per token (one warp each), then Algorithm 1, redundantly in every CTA ----
    for (int i = tid; i < T_ * E; i += kStreamConsumers) s_z[i] = a.logits[i];
    asm volatile("bar.sync 1, 256;" ::: "memory");
    topk_softmax_block(s_z, T_, E, k, s_ids, s_w, s_selz, kStreamConsumers, 1);
#ifndef WISP_PROBE_TIMELINE
    stamp(1);
#endif
    if (writer && tid < T_ * k) {
      const size_t off = (size_t)l * a.max_tokens * k;
      a.ids[off + tid] = s_ids[tid];
      a.topw[off + tid] = s_w[tid];
    }
    {
      PlanArgs pa;
      pa.ids = s_ids; pa.n_pairs = T_ * k; pa.E = E; pa.C = C; pa.policy = a.policy; pa.layer = l;
      pa.st = st; pa.plan = pp; pa.host_plan = nullptr;
      pa.trace = a.trace; pa.trace_ctr = a.trace_ctr; pa.trace_cap = a.trace_cap; pa.trace_on = a.trace_on;
      pa.track = a.track; pa.build_pairs = 1; pa.wave_order = a.wave_order;
      plan_compute<kPersistMaxExperts>(pa, sh, writer, 1);
    }
    if (tid == 0) mbar_arrive(smem_u32(&s_plan_ready));                      // the producer may start streaming
    stamp(2);
    if (l + 1 < a.layer_hi) {
      // While the ring fills: the next layer's residency state -> smem (stable until that layer's own plan phase)
      // and its router rows -> smem (TMA), so the serial router -> top-k -> plan chain of layer l+1 starts from warm data.
      plan_load<kPersistMaxExperts>(sh, layer_state_of(a, l + 1), E, C);
      stage_router_rows(l + 1);
    }
    stamp(3);

    // ---- phases G, D per wave ----
    sa.layer = l;
    sa.master = a.fused ? a.masters[l] : nullptr;
    const int n_waves = pl.hdr[0], nR = pl.hdr[1];
    const int miss_cls = pl.hdr[2] > 0 ? 3 : 0;                              // layers with misses are timed apart
#ifdef WISP_PROBE_TIMELINE
    mute = miss_cls != 0;
    if (timing && !mute) a.phase_ns[kPersistPhases] += 1;
#else
    if (timing) a.phase_ns[kPersistPhases + (miss_cls ? 1 : 0)] += 1;
#endif
    for (int w = 0; w < n_waves; ++w) {
      const int lo = w * C, nw = min(nR, lo + C) - lo;
      {
        const long long U = (long long)nw * ggu.upe;
        sa.operand = x_l; sa.result = a.act; sa.out_ld = dff;
#ifdef WISP_PROBE_TIMELINE   // profiling probe only: slot 1 = wait for the first G tile, 3 = barrier C, 7 = first D tile, 8 = barrier D
        u64* cta_probe = a.phase_ns + 16 + blockIdx.x * 8;                   // per-CTA absolute times of the last layer
        if (tid == 0 && a.phase_ns && l == a.layer_hi - 1) cta_probe[0] = globaltimer_ns();
        if (tid == 0) mbar_wait(ring.full0 + 8u * rp.s, rp.ph);
        if (tid == 0 && a.phase_ns && l == a.layer_hi - 1) { cta_probe[1] = globaltimer_ns(); cta_probe[5] = (u64)((int)(U * (blockIdx.x + 1) / gridDim.x) - (int)(U * blockIdx.x / gridDim.x)); }
        stamp(1);
#endif
        stream_consume<T, 0, NP>(sa, ggu, ring, rp, lo, (int)(U * blockIdx.x / gridDim.x), (int)(U * (blockIdx.x + 1) / gridDim.x),
                                 s_red, par, 2);
      }
#ifdef WISP_PROBE_TIMELINE
      if (tid == 0 && a.phase_ns && l == a.layer_hi - 1) a.phase_ns[16 + blockIdx.x * 8 + 2] = globaltimer_ns();
      stamp(4);
      grid_barrier(a.gbar, gen, a.err);
      if (tid == 0 && a.phase_ns && l == a.layer_hi - 1) a.phase_ns[16 + blockIdx.x * 8 + 3] = globaltimer_ns();
      stamp(3);
      if (tid == 0) mbar_wait(ring.full0 + 8u * rp.s, rp.ph);
      stamp(7);
#else
      grid_barrier(a.gbar, gen, a.err);                                      // C: act rows of this wave complete
      stamp(4 + miss_cls);
#endif
      {
        const long long U = (long long)nw * gdn.upe;
        sa.operand = a.act; sa.result = a.ystage; sa.out_ld = d;
        stream_consume<T, 1, NP>(sa, gdn, ring, rp, lo, (int)(U * blockIdx.x / gridDim.x), (int)(U * (blockIdx.x + 1) / gridDim.x),
                                 s_red, par, 2);
      }
#ifdef WISP_PROBE_TIMELINE
      if (tid == 0 && a.phase_ns && l == a.layer_hi - 1) a.phase_ns[16 + blockIdx.x * 8 + 4] = globaltimer_ns();
      stamp(5);
      grid_barrier(a.gbar, gen, a.err);
      stamp(8);
#else
      grid_barrier(a.gbar, gen, a.err);                                      // D: ystage complete; slots of the wave free
      stamp(5 + miss_cls);
#endif
    }

    // ---- phase X: ordered combine (+ residual), split over the grid ----
    // x_{l+1} goes through global memory and one grid barrier, then every CTA reloads it into its xs.  (Recomputing the whole
    // x_{l+1} in every CTA saves the barrier but makes 148 CTAs read the same T x 64 KiB of ystage from L2: measured slower, 490 vs
    // 500 tokens/s at one token, 674 vs 764 at four.)
    {
      const int n = T_ * d;
      const bool last = l == a.layer_hi - 1;
      T* xg = reinterpret_cast<T*>(last ? a.out : a.xbuf[(l - a.layer_lo) & 1]);
      // 4 consecutive elements per thread; the ystage loads of up to 8 ranks are issued together (one L2 round trip),
      // the sum itself is combine_elem's: fmaf in rank order from 0.f, per element.
      for (int v4 = (int)blockIdx.x * kStreamConsumers + tid; v4 < n / 4; v4 += (int)gridDim.x * kStreamConsumers) {
        const int idx = v4 * 4, t = idx / d, j = idx % d;
        float acc[4] = {0.f, 0.f, 0.f, 0.f};
        for (int i0 = 0; i0 < k; i0 += 8) {
          float4 y[8];
#pragma unroll
          for (int u = 0; u < 8; ++u)
            if (i0 + u < k) y[u] = *reinterpret_cast<const float4*>(a.ystage + ((size_t)t * k + i0 + u) * d + j);
#pragma unroll
          for (int u = 0; u < 8; ++u)
            if (i0 + u < k) {
              const float w = s_w[t * k + i0 + u];
              acc[0] = fmaf(w, y[u].x, acc[0]); acc[1] = fmaf(w, y[u].y, acc[1]);
              acc[2] = fmaf(w, y[u].z, acc[2]); acc[3] = fmaf(w, y[u].w, acc[3]);
            }
        }
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          const T o = from_f32<T>(acc[c]);
          xg[idx + c] = a.residual ? from_f32<T>(to_f32<T>(xs[idx + c]) + to_f32<T>(o)) : o;
        }
      }
      if (!last) {
        grid_barrier(a.gbar, gen, a.err);                                    // E: x_{l+1} complete in global memory
        const uint4* src = reinterpret_cast<const uint4*>(xg);
        uint4* dst = reinterpret_cast<uint4*>(xs);
        for (int i = tid; i < n * (int)sizeof(T) / 16; i += kStreamConsumers) dst[i] = src[i];
      }
    }
    asm volatile("bar.sync 1, 256;" ::: "memory");                           // xs complete in this CTA
    stamp(6);
    mute = false;
  }
}

}  // namespace wisp
