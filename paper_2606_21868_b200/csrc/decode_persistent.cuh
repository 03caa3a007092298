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
//   phase X  combine (+ residual)     distributed over all CTAs, rank order (combine_elem)        -> barrier E
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
constexpr int kPersistPhases = 5;           // timing classes: router, plan, gate_up, down, combine
constexpr unsigned kGridBarrierSpinLimit = 1u << 26;

struct PersistArgs {
  int L, E, k, d, dff, T, C, policy;
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
    __threadfence();                       // cumulative: the CTA's writes ordered before the arrival
    atomicAdd(ctr, 1u);
    unsigned seen, spins = 0;
    do {
      asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(ctr) : "memory");
      if (++spins > kGridBarrierSpinLimit) { *err = 1; break; }
    } while (seen < gen);
    __threadfence();                       // gpu-scope fence: also invalidates this SM's L1
  }
  asm volatile("bar.sync 1, 256;" ::: "memory");
}

template <typename T, int NP>
__global__ void __launch_bounds__(kStreamThreads, 1) decode_persistent_kernel(const PersistArgs a, const StreamGeom ggu,
                                                                              const StreamGeom gdn, int n_stages, int stage_stride) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  __shared__ __align__(8) unsigned long long s_full[kStreamMaxStages], s_empty[kStreamMaxStages], s_plan_ready;
  __shared__ float s_red[2 * (kStreamConsumers / 32) * StreamBatch<NP>::NVAL];
  __shared__ PlanShared<kPersistMaxExperts> sh;
  __shared__ PersistPlan pl;
  __shared__ float s_z[NP * kPersistMaxExperts];   // logits, rows packed E apart
  __shared__ float s_selz[NP * kMaxTopK];
  __shared__ int s_ids[NP * kMaxTopK];
  __shared__ float s_w[NP * kMaxTopK];

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  Ring ring;
  ring.stage0 = smem_u32(smem_raw); ring.full0 = smem_u32(s_full); ring.empty0 = smem_u32(s_empty);
  ring.NS = n_stages; ring.stride = stage_stride;
  if (tid == 0) {
    mbar_init(smem_u32(&s_plan_ready), 1);
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
  auto stamp = [&](int phase) {
    if (timing) { const u64 t = globaltimer_ns(); a.phase_ns[phase] += t - t_prev; t_prev = t; }
  };
  unsigned gen = 0;
  int par = 0;
  plan_load<kPersistMaxExperts>(sh, layer_state_of(a, a.layer_lo), E, C);
  for (int l = a.layer_lo; l < a.layer_hi; ++l) {
    const int rel = l - a.layer_lo;
    const T* x_l = reinterpret_cast<const T*>(rel == 0 ? a.x_in : a.xbuf[(rel - 1) & 1]);
    T* x_next = reinterpret_cast<T*>(l == a.layer_hi - 1 ? a.out : a.xbuf[rel & 1]);
    const LayerState st = layer_state_of(a, l);

    // ---- phase R: router logits (this layer's residency state is already in `sh`, its router rows in L2) ----
    {
      const T* wr = reinterpret_cast<const T*>(a.router_w) + (size_t)l * E * d;
      const float* bias = a.router_bias + (size_t)l * E;
      for (int e = warp * gridDim.x + blockIdx.x; e < E; e += (kStreamConsumers / 32) * gridDim.x)
        for (int t0 = 0; t0 < T_; t0 += kRouterTokTile)
          router_row_warp<T>(x_l, wr + (size_t)e * d, bias[e], a.logits, e, t0, min(kRouterTokTile, T_ - t0), E, d, lane);
    }
    grid_barrier(a.gbar, gen, a.err);                                        // B: logits complete
    stamp(0);

    // ---- phase P: top-k + softmax per token (one warp each), then Algorithm 1, redundantly in every CTA ----
    for (int i = tid; i < T_ * E; i += kStreamConsumers) s_z[i] = a.logits[i];
    asm volatile("bar.sync 1, 256;" ::: "memory");
    topk_softmax_block(s_z, T_, E, k, s_ids, s_w, s_selz, kStreamConsumers, 1);
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
      pa.track = a.track; pa.build_pairs = 1;
      plan_compute<kPersistMaxExperts>(pa, sh, writer, 1);
    }
    if (tid == 0) mbar_arrive(smem_u32(&s_plan_ready));                      // the producer may start streaming
    if (l + 1 < a.layer_hi) {
      // While the ring fills: the next layer's residency state -> smem (stable until that layer's own plan phase)
      // and its router rows -> L2, so the serial router -> top-k -> plan chain of layer l+1 starts from warm data.
      plan_load<kPersistMaxExperts>(sh, layer_state_of(a, l + 1), E, C);
      const char* wr = a.router_w + (size_t)(l + 1) * E * d * sizeof(T);
      for (int e = warp * gridDim.x + blockIdx.x; e < E; e += (kStreamConsumers / 32) * gridDim.x)
        if (lane == 0) l2_prefetch(wr + (size_t)e * d * sizeof(T), (uint32_t)(d * sizeof(T)));
    }
    stamp(1);

    // ---- phases G, D per wave ----
    sa.layer = l;
    sa.master = a.fused ? a.masters[l] : nullptr;
    const int n_waves = pl.hdr[0], nR = pl.hdr[1];
    for (int w = 0; w < n_waves; ++w) {
      const int lo = w * C, nw = min(nR, lo + C) - lo;
      {
        const long long U = (long long)nw * ggu.upe;
        sa.operand = x_l; sa.result = a.act; sa.out_ld = dff;
        stream_consume<T, 0, NP>(sa, ggu, ring, rp, lo, (int)(U * blockIdx.x / gridDim.x), (int)(U * (blockIdx.x + 1) / gridDim.x),
                                 s_red, par, 2);
      }
      grid_barrier(a.gbar, gen, a.err);                                      // C: act rows of this wave complete
      stamp(2);
      {
        const long long U = (long long)nw * gdn.upe;
        sa.operand = a.act; sa.result = a.ystage; sa.out_ld = d;
        stream_consume<T, 1, NP>(sa, gdn, ring, rp, lo, (int)(U * blockIdx.x / gridDim.x), (int)(U * (blockIdx.x + 1) / gridDim.x),
                                 s_red, par, 2);
      }
      grid_barrier(a.gbar, gen, a.err);                                      // D: ystage complete; slots of the wave free
      stamp(3);
    }

    // ---- phase X: ordered combine (+ residual), distributed over the grid ----
    {
      const int n = T_ * d;
      for (int idx = blockIdx.x * kStreamConsumers + tid; idx < n; idx += gridDim.x * kStreamConsumers) {
        const int t = idx / d, j = idx % d;
        T o, xn;
        combine_elem<T>(a.ystage, s_w, t, j, d, k, a.residual ? x_l[idx] : from_f32<T>(0.f), o, xn);
        x_next[idx] = a.residual ? xn : o;
      }
    }
    if (l + 1 < a.layer_hi) grid_barrier(a.gbar, gen, a.err);                // E: x_{l+1} complete
    stamp(4);
  }
}

}  // namespace wisp
